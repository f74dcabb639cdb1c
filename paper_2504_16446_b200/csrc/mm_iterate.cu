// mm_iterate.cu — NEXT-3: a regularised Nesterov iteration that stays on the device, with the relative-change stop
// rule (MITRA = gradient descent + Nesterov momentum + arbitrary regularisers, SIGTT stops on the
// relative change of the loss; the asynchronous pipelines keep the whole loop on the GPU).
// Reading S25 fixes the formulas; the oracle's `iterate` is the same loop in numpy.
//
// Everything an iteration needs is enqueued on one stream: look-ahead point, fused loss + gradient
// (mm_loss_gradient), Laplacian and L2 terms, total loss, update.  The loss history and the stop flag live in device
// memory; the host reads ONE 4-byte flag every `check_every` iterations and nothing else crosses the bus.
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "mm_internal.h"

namespace {

// y = c + m v on channels < K (pad channels of y are written 0: they are inputs of the forward model only in name)
__global__ void lookahead_kernel(float *__restrict__ y, const float *__restrict__ c, const float *__restrict__ v, float m, long long n,
                                 int ldk, int K)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) y[i] = (int)(i % ldk) < K ? fmaf(m, v[i], c[i]) : 0.f;
}

// out += sum over channels < K of x^2 (fp64, one atomic per block)
__global__ void __launch_bounds__(256) sumsq_kernel(const float *__restrict__ x, long long n, int ldk, int K, double *__restrict__ out)
{
    double s = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        if ((int)(i % ldk) < K) { const double t = x[i]; s = fma(t, t, s); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __shared__ double red[8];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; w++) t += red[w];
        atomicAdd(out, t);
    }
}

// L_k = data term + mu_lap/2 ||Lap y||^2 + mu_l2/2 ||y||^2; stop flag after every check_every-th iteration:
// |L_k - L_{k-1}| <= tol |L_k|
__global__ void loss_total_kernel(double *__restrict__ losses, int k, const double *__restrict__ terms /*data, ss_lap, ss_l2*/,
                                  float mu_lap, float mu_l2, double tol, int check_every, int *__restrict__ flag)
{
    const double L = terms[0] + 0.5 * (double)mu_lap * terms[1] + 0.5 * (double)mu_l2 * terms[2];
    losses[k] = L;
    if (k >= 1 && (k + 1) % check_every == 0 && fabs(L - losses[k - 1]) <= tol * fabs(L)) *flag = 1;
}

// g = grad + mu_lap Lap(Lap y) + mu_l2 y;  v <- m v - eta g;  c <- c + v   (channels < K only)
__global__ void iterate_update_kernel(float *__restrict__ c, float *__restrict__ v, const float *__restrict__ grad,
                                      const float *__restrict__ lap2, const float *__restrict__ y, float mu_lap, float mu_l2, float eta,
                                      float m, long long n, int ldk, int K)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || (int)(i % ldk) >= K) return;
    float g = grad[i];
    if (lap2) g = fmaf(mu_lap, lap2[i], g);
    if (mu_l2 != 0.f) g = fmaf(mu_l2, y[i], g);
    const float vn = fmaf(m, v[i], -eta * g);
    v[i] = vn;
    c[i] += vn;
}

}  // namespace

extern "C" mm_status mm_iterate(const mm_geometry *g, const float *B, int32_t K, int32_t ldk, int32_t D, const float *data,
                                const float *weights, const mm_iterate_params *p, float *c, float *v, double *losses,
                                int32_t *n_iter, void *stream)
{
    if (!g || !B || !data || !p || !c || !v || !losses || !n_iter) { mm_set_error("mm_iterate: NULL argument"); return MM_ERR_NULL; }
    if (K < 1 || ldk < K || D < 1 || D > MM_MAX_D) { mm_set_error("mm_iterate: need 1 <= K <= ldk, 1 <= D <= MM_MAX_D"); return MM_ERR_SHAPE; }
    if (p->max_iter < 1 || p->check_every < 1) { mm_set_error("mm_iterate: max_iter and check_every must be positive"); return MM_ERR_VALUE; }
    if (!(p->eta > 0.f) || !(p->momentum >= 0.f) || !(p->mu_laplacian >= 0.f) || !(p->mu_l2 >= 0.f)) {
        mm_set_error("mm_iterate: need eta > 0 and non-negative momentum and regularisation weights");
        return MM_ERR_VALUE;
    }
    *n_iter = 0;
    cudaStream_t st = (cudaStream_t)stream;
    const long long nvox = (long long)g->shape[0] * g->shape[1] * g->shape[2];
    const long long n = nvox * ldk;
    const size_t vol_bytes = ((size_t)n * sizeof(float) + 255) & ~(size_t)255;
    const size_t sino_bytes = ((size_t)g->P * g->J * g->Kd * D * sizeof(float) + 255) & ~(size_t)255;
    const bool lap = p->mu_laplacian > 0.f;
    // scratch (stream-ordered, from the library's pool): look-ahead point, gradient, [Lap y, Lap Lap y], wr, 3 doubles + flag
    char *base = nullptr;
    const size_t total = (lap ? 4 : 2) * vol_bytes + sino_bytes + 256;
    cudaError_t e = mm_scratch_alloc((void **)&base, total, st);
    if (e != cudaSuccess) { mm_set_error(std::string("mm_iterate: scratch: ") + cudaGetErrorString(e)); cudaGetLastError(); return MM_ERR_ALLOC; }
    float *y = (float *)base, *grad = (float *)(base + vol_bytes);
    float *lap1 = lap ? (float *)(base + 2 * vol_bytes) : nullptr, *lap2 = lap ? (float *)(base + 3 * vol_bytes) : nullptr;
    float *wr = (float *)(base + (lap ? 4 : 2) * vol_bytes);
    double *terms = (double *)((char *)wr + sino_bytes);
    int *flag = (int *)(terms + 4);
    const unsigned nb = (unsigned)((n + 255) / 256);
    const unsigned rb = (unsigned)(nb < 148u * 8u ? nb : 148u * 8u);          // reduction: a few blocks per SM, grid-stride
    mm_status rc = MM_OK;
    int done = 0, h_flag = 0;
    auto launch_ok = [&](const char *what) {
        const cudaError_t le = cudaGetLastError();
        if (le != cudaSuccess) { mm_set_error(std::string("mm_iterate: ") + what + ": " + cudaGetErrorString(le)); rc = MM_ERR_CUDA; return false; }
        return true;
    };
    if (cudaMemsetAsync(flag, 0, sizeof(int), st) != cudaSuccess) { launch_ok("memset"); rc = MM_ERR_CUDA; }
    for (int k = 0; k < p->max_iter && rc == MM_OK; k++) {
        lookahead_kernel<<<nb, 256, 0, st>>>(y, c, v, p->momentum, n, ldk, K);
        if (!launch_ok("lookahead_kernel")) break;
        rc = mm_loss_gradient(g, B, y, K, ldk, D, data, weights, grad, terms, wr, st);      // terms[0] = data term
        if (rc != MM_OK) break;
        if (cudaMemsetAsync(terms + 1, 0, 2 * sizeof(double), st) != cudaSuccess) { launch_ok("memset"); rc = MM_ERR_CUDA; break; }
        if (lap) {
            rc = mm_laplacian(g, y, K, ldk, lap1, st);
            if (rc == MM_OK) rc = mm_laplacian(g, lap1, K, ldk, lap2, st);
            if (rc != MM_OK) break;
            sumsq_kernel<<<rb, 256, 0, st>>>(lap1, n, ldk, K, terms + 1);
            if (!launch_ok("sumsq_kernel")) break;
        }
        if (p->mu_l2 > 0.f) {
            sumsq_kernel<<<rb, 256, 0, st>>>(y, n, ldk, K, terms + 2);
            if (!launch_ok("sumsq_kernel")) break;
        }
        loss_total_kernel<<<1, 1, 0, st>>>(losses, k, terms, p->mu_laplacian, p->mu_l2, p->tol, p->check_every, flag);
        if (!launch_ok("loss_total_kernel")) break;
        iterate_update_kernel<<<nb, 256, 0, st>>>(c, v, grad, lap2, y, p->mu_laplacian, p->mu_l2, p->eta, p->momentum, n, ldk, K);
        if (!launch_ok("iterate_update_kernel")) break;
        mm_note_launches(3 + (lap ? 1 : 0) + (p->mu_l2 > 0.f ? 1 : 0));     // look-ahead, total, update (+ reductions)
        done = k + 1;
        if (p->tol > 0.0 && k >= 1 && (k + 1) % p->check_every == 0) {                  // the only host round trip: 4 bytes
            if (cudaMemcpyAsync(&h_flag, flag, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaStreamSynchronize(st) != cudaSuccess) { launch_ok("flag read"); rc = MM_ERR_CUDA; break; }
            if (h_flag) break;
        }
    }
    mm_scratch_free(base, st);
    *n_iter = done;
    return rc;
}
