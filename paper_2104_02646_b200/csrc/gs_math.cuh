// gs_math.cuh -- fp32 3-vector helpers for the CUDA path (device only).
#pragma once
#include <cuda_runtime.h>

namespace gs {

struct vec3 {
    float x, y, z;
    __host__ __device__ __forceinline__ vec3() {}
    __host__ __device__ __forceinline__ vec3(float a, float b, float c) : x(a), y(b), z(c) {}
    __host__ __device__ __forceinline__ explicit vec3(const float4 &v) : x(v.x), y(v.y), z(v.z) {}
};

__host__ __device__ __forceinline__ vec3 operator+(vec3 a, vec3 b) { return vec3(a.x + b.x, a.y + b.y, a.z + b.z); }
__host__ __device__ __forceinline__ vec3 operator-(vec3 a, vec3 b) { return vec3(a.x - b.x, a.y - b.y, a.z - b.z); }
__host__ __device__ __forceinline__ vec3 operator-(vec3 a) { return vec3(-a.x, -a.y, -a.z); }
__host__ __device__ __forceinline__ vec3 operator*(float s, vec3 a) { return vec3(s * a.x, s * a.y, s * a.z); }
__host__ __device__ __forceinline__ vec3 operator*(vec3 a, float s) { return vec3(s * a.x, s * a.y, s * a.z); }
__host__ __device__ __forceinline__ vec3 &operator+=(vec3 &a, vec3 b) { a.x += b.x; a.y += b.y; a.z += b.z; return a; }
__host__ __device__ __forceinline__ vec3 &operator-=(vec3 &a, vec3 b) { a.x -= b.x; a.y -= b.y; a.z -= b.z; return a; }
__host__ __device__ __forceinline__ float dot(vec3 a, vec3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__host__ __device__ __forceinline__ vec3 cross(vec3 a, vec3 b) {
    return vec3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
// a + s*b
__host__ __device__ __forceinline__ vec3 madd(vec3 a, float s, vec3 b) { return vec3(fmaf(s, b.x, a.x), fmaf(s, b.y, a.y), fmaf(s, b.z, a.z)); }
__host__ __device__ __forceinline__ vec3 zero3() { return vec3(0.f, 0.f, 0.f); }

}  // namespace gs
