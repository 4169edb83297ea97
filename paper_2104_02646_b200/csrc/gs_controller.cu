// gs_controller.cu -- the open-loop MPC controller that produces the activation schedule, and dL/dW.
//
// PAPER.md:777 (appendix "MPC Controller Architecture"): "we generate N phase-shifted sinusoidal signals which are passed to a
// fully-connected layer (zero-bias), and a final activation layer.  The output is a vector of per-element activation
// values"; one fully connected layer and a tanh, 8 signals.  DESIGN.md reading A23b:
//     s_i(t) = sin(omega t + 2 pi i / N),   act_e(t_f) = A tanh(sum_i W[e, i] s_i(t_f)),   t_f = f frame_dt
//     dL/dW[e, i] = sum_f dL/dact_e(t_f) A (1 - tanh^2(y_e(t_f))) s_i(t_f)
// Layouts (caller order): W, dL/dW [E][count][N]; act, dL/dact [F][E][count] -- what gs_set_actuation takes and
// gs_actuation_grads writes.  The signal table [F][N] is built in shared memory by every CTA (phase in fp64, reduced modulo
// 2 pi before the fp32 sine); the layer is a handful of FMAs per output.  Nothing here is shared with the oracle.
#include <cstdint>

#include "gs_internal.h"

namespace gs {

constexpr int kCtlTable = 8192;  // signal-table entries staged at once (32 KB)

__device__ __forceinline__ float ctl_signal(int i, int n, double omega_t) {
    const double two_pi = 6.283185307179586476925286766559;
    const double a = fmod(omega_t + two_pi * (double)i / (double)n, two_pi);
    return sinf((float)a);
}
// frames [f0, f1) of the table into shared memory
__device__ __forceinline__ void ctl_table(float *s, int f0, int f1, int n, float omega, float frame_dt) {
    for (int q = threadIdx.x; q < (f1 - f0) * n; q += blockDim.x) {
        const int f = f0 + q / n, i = q % n;
        s[q] = ctl_signal(i, n, (double)omega * ((double)f * (double)frame_dt));
    }
    __syncthreads();
}

// one thread per (env, element), all frames
__global__ void __launch_bounds__(256) k_controller_fwd(int F, size_t EM, int n, float omega, float frame_dt, float amp, const float *__restrict__ W,
                                                         float *__restrict__ act) {
    __shared__ float s[kCtlTable];
    const size_t em = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int fc = kCtlTable / n;
    for (int f0 = 0; f0 < F; f0 += fc) {
        const int f1 = min(F, f0 + fc);
        ctl_table(s, f0, f1, n, omega, frame_dt);
        if (em < EM)
            for (int f = f0; f < f1; f++) {
                float y = 0.f;
                for (int i = 0; i < n; i++) y = fmaf(W[em * n + i], s[(f - f0) * n + i], y);
                act[(size_t)f * EM + em] = amp * tanhf(y);
            }
        __syncthreads();
    }
}

// one thread per (env, element, signal): y is rebuilt per frame (n FMAs)
__global__ void __launch_bounds__(256) k_controller_adj(int F, size_t EM, int n, float omega, float frame_dt, float amp, const float *__restrict__ W,
                                                         const float *__restrict__ g_act, float *__restrict__ g_W) {
    __shared__ float s[kCtlTable];
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x, em = q / n;
    const int i = (int)(q - em * n);
    const bool on = em < EM;
    const int fc = kCtlTable / n;
    float acc = 0.f;
    for (int f0 = 0; f0 < F; f0 += fc) {
        const int f1 = min(F, f0 + fc);
        ctl_table(s, f0, f1, n, omega, frame_dt);
        if (on)
            for (int f = f0; f < f1; f++) {
                float y = 0.f;
                for (int k = 0; k < n; k++) y = fmaf(W[em * n + k], s[(f - f0) * n + k], y);
                const float th = tanhf(y);
                acc = fmaf(g_act[(size_t)f * EM + em] * amp * (1.0f - th * th), s[(f - f0) * n + i], acc);
            }
        __syncthreads();
    }
    if (on) g_W[q] = acc;
}

}  // namespace gs

using namespace gs;

static int ctl_check(int n_frames, int n_envs, int count, int n_signals, float frame_dt, const void *a, const void *b) {
    if (n_frames < 1 || n_envs < 1 || count < 1 || n_signals < 1 || n_signals > kCtlTable) { set_error("controller: n_frames, n_envs, count >= 1 and 1 <= n_signals <= %d", kCtlTable); return GS_EINVAL; }
    if (!(frame_dt > 0.f)) { set_error("controller: frame_dt must be positive"); return GS_EINVAL; }
    if (!a || !b) { set_error("controller: null array"); return GS_EINVAL; }
    return GS_OK;
}

extern "C" int gs_controller_schedule(int n_frames, int n_envs, int count, int n_signals, float omega, float frame_dt, float amplitude, const float *d_W,
                                      float *d_act, gs_stream stream) {
    int rc = ctl_check(n_frames, n_envs, count, n_signals, frame_dt, d_W, d_act);
    if (rc != GS_OK) return rc;
    const size_t EM = (size_t)n_envs * count;
    k_controller_fwd<<<(unsigned)((EM + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n_frames, EM, n_signals, omega, frame_dt, amplitude, d_W, d_act);
    count_launch();
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? GS_OK : cuda_fail(e, "k_controller_fwd");
}

extern "C" int gs_controller_grads(int n_frames, int n_envs, int count, int n_signals, float omega, float frame_dt, float amplitude, const float *d_W,
                                   const float *d_g_act, float *d_g_W, gs_stream stream) {
    int rc = ctl_check(n_frames, n_envs, count, n_signals, frame_dt, d_W, d_g_act);
    if (rc == GS_OK && !d_g_W) { set_error("controller: null array"); rc = GS_EINVAL; }
    if (rc != GS_OK) return rc;
    const size_t EM = (size_t)n_envs * count, Q = EM * n_signals;
    k_controller_adj<<<(unsigned)((Q + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n_frames, EM, n_signals, omega, frame_dt, amplitude, d_W, d_g_act, d_g_W);
    count_launch();
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? GS_OK : cuda_fail(e, "k_controller_adj");
}
