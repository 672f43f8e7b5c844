// tb_whiten.cuh -- front-end whitening once per series ("Fourier
// birdie zapping, ..., Fourier de-reddening", L660; the paper gives no formulas: reading G25 of
// DESIGN.md section 3).  Run by tb_plan_create / tb_plan_set_series when opts.whiten is set:
//
//   X = D2Z(x)                                   (cuFFT, one length-N transform, in fp64)
//   m_b = exact median of |X_k|^2 over each block of W bins        k_whiten_medians
//   X'_k = X_k / sqrt(m(k) / ln2) / sqrt(N), m(k) interpolated linearly between block centres
//          (G15); X'_0 = X'_{N/2} = 0; zapped ranges = 0            k_whiten_apply
//   x' = Z2D(X')                                 (cuFFT; the 1/sqrt(N) above makes it unit variance)
//   kappa = ln2 / mean_b(median of the interbinned spectrum of x' over block b)
//
// The two transforms run in double precision: this is once per series (0.4 ms at 2^23, against 27 ms
// for a 512-template bank), and a single-precision R2C of a RED series loses its top bins, which
// the real-to-complex unpack forms as small differences of the huge bins mirrored from the bottom
// of the spectrum (2e-4 of the baseline in the red-noise parity test).
//
// after which every template is normalised by the constant kappa instead of its own block medians
// (a6 leaves the per-template loop; the spectrum kernels' WHITE variants).
#pragma once
#include "tb_kernels.cuh"

namespace tb {

constexpr int WH_WARPS = 8;

// one warp = one block of W raw powers |X_k|^2 (X: cuFFT R2C output, N/2+1 values) -> med[block]
template <int W>
__global__ void __launch_bounds__(WH_WARPS * 32) k_whiten_medians(const double2* __restrict__ X, int nblk, float* __restrict__ med)
{
    constexpr int VPT = W / 32;
    __shared__ float s_cand[WH_WARPS][med_scratch_floats<W>()];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int blk = blockIdx.x * WH_WARPS + wid;
    if (blk >= nblk) return;
    const double2* __restrict__ xb = X + (size_t)blk * W;
    float p[VPT];
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
        const double2 v = xb[i * 32 + lane];
        p[i] = (float)fma(v.y, v.y, v.x * v.x);
    }
    const float m = warp_median<W>(p, s_cand[wid], lane, nullptr);
    if (lane == 0) med[blk] = m;
}

// X'_k = X_k * sqrt(ln2 / m(k)) * inv_sqrt_n, in place over the N/2+1 values of X
__global__ void __launch_bounds__(256)
k_whiten_apply(double2* __restrict__ X, int nb, int log2w, int nblk, const float* __restrict__ med, double inv_sqrt_n,
               const uint2* __restrict__ zap, int n_zap)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > nb) return;
    double2 v = make_double2(0.0, 0.0);
    if (k > 0 && k < nb) {
        // baseline between the block centres c_b = b W + (W - 1)/2, flat outside (G15)
        // in integers: t = 2k - (W - 1) = twice the offset from centre 0; block b0 = floor(t / 2W), fraction exact in fp32
        const int t = 2 * k - ((1 << log2w) - 1);
        int b0 = t >> (log2w + 1);
        float fr = (float)(t - (b0 << (log2w + 1))) / (float)(2 << log2w);
        if (t <= 0) { b0 = 0; fr = 0.f; }
        if (b0 >= nblk - 1) { b0 = nblk - 1; fr = 0.f; }
        const float ma = __ldg(med + b0), mb = __ldg(med + min(b0 + 1, nblk - 1));
        const float m = fmaf(fr, mb - ma, ma);
        if (m > 0.f) {
            const double s = sqrt(0.69314718055994530942 / (double)m) * inv_sqrt_n;
            const double2 x = X[k];
            v = make_double2(x.x * s, x.y * s);
        }
        for (int z = 0; z < n_zap; ++z) {
            const uint2 r = __ldg(zap + z);
            if ((unsigned)k >= r.x && (unsigned)k < r.y) v = make_double2(0.0, 0.0);
        }
    }
    X[k] = v;
}

__global__ void __launch_bounds__(256) k_f32_to_f64(const float* __restrict__ x, double* __restrict__ y, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) y[i] = (double)x[i];
}
__global__ void __launch_bounds__(256) k_f64_to_f32(const double* __restrict__ x, float* __restrict__ y, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) y[i] = (float)x[i];
}

}  // namespace tb
