// tb_kernels.cuh -- device code of libtb (sm_100a).  See include/tb.h for the boundary and
// DESIGN.md sections 6-7 for the data layout, the byte model and the roofline of each kernel.
//
// Nothing on this path is a dense contraction, so no tensor cores: the kernels are bound by
// HBM (streaming 128-bit loads/stores), by the fp64 pipe (delay model) or by instruction issue
// (median select, harmonic sum).  Citations: PAPER.md line numbers; G<n> = DESIGN.md readings.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tb {

// ---------------------------------------------------------------------------------------------
// per-template constants (step a1), computed on the host in extended precision
// ---------------------------------------------------------------------------------------------
struct TmplDev {
    double c_hi, c_lo;   // orbital turns per sample tsamp/P_orb as a double-double
    double w;            // radians per sample 2*pi*tsamp/P_orb
    double phi0;         // initial orbital phase reduced to [0, 2*pi)
    double A, B;         // (tau/tsamp) sin(omega), (tau/tsamp) sqrt(1-e^2) cos(omega)   (eq A1)
    double ecc;          // e
    double d0;           // zero offset in samples: A cos E0 + B sin E0 at M = phi0      (L675, L682-692)
    int32_t log2h;       // Hermite knot spacing h = 2^log2h samples (0: every sample is a knot)
    int32_t circular;    // 1: e == 0, E = M (no Kepler solve)
    uint32_t id;         // template id reported in the candidates (first_template_id + index in the caller's array)
    uint32_t pad;
};

// ELL7 approximate-orbit mode (reading G26; eqs 15-16,
// App. B): cos E = sum C_k(e) cos kM, sqrt(1-e^2) sin E = sum S_k(e) sin kM, k = 1..7
// (C_0 and the -e of eq A1 are constants and cancel against the zero offset).
struct EllCoef {
    double c[8];         // c[k-1] = C_k(e), k = 1..7 (c[7] unused)
    double s[8];         // s[k-1] = S_k(e)
};

struct FoldParams {
    float    thr[5];     // power threshold T_L per fold, +inf for folds not requested
    float    mu[5];      // mu_n, n = 2^L
    float    inv_s[5];   // 1/s_n
    uint32_t lo[5];      // lowest bin of fold L: min(k_lo 2^L, Nb), made on the host in 64 bits (G20)
};

struct Candidate {       // == tb_candidate
    uint32_t template_id, fold, bin;
    float    power, sigma;
    uint32_t pad;
};

constexpr int RS_THREADS = 256;      // resampler CTA
constexpr int RS_TILE    = 4096;     // output samples per CTA
constexpr int RS_MAXSEG  = 512;      // Hermite segments held in shared memory at once
constexpr int SP_WARPS   = 8;        // spectrum/median CTA = 8 warps, one median block per warp

// ---------------------------------------------------------------------------------------------
// a2: exact delay (in samples, zero offset removed) and its per-sample slope at sample j.
//   phase in turns u = frac(j * tsamp/P_orb) from a double-double product, so that the mean
//   anomaly M = 2 pi u + phi0 carries ~1e-17 rad of error instead of ulp(Omega t) (DESIGN.md
//   section 6.1: index parity error budget).  E from Newton's method on E - e sin E = M
//   (eq 3; Alg. 1; G9), delay from eq A1 (L666).
// ---------------------------------------------------------------------------------------------
//   ell != nullptr: the ELL7 series instead of the Kepler solve (then t.A = (tau/tsamp) sin(omega),
//   t.B = (tau/tsamp) cos(omega): the S-series carries the sqrt(1-e^2)); cos kM, sin kM by the
//   Chebyshev recurrence from one sincos.
__device__ __forceinline__ void delay_knot(const TmplDev& t, int j, double& val, double& slope, const EllCoef* __restrict__ ell = nullptr)
{
    const double TWO_PI_HI = 6.283185307179586232;      // fl(2 pi)
    const double TWO_PI_LO = 2.449293598294706414e-16;  // 2 pi - fl(2 pi)
    const double jd  = (double)j;
    const double p   = jd * t.c_hi;
    double lo        = fma(jd, t.c_hi, -p);              // exact product error
    lo               = fma(jd, t.c_lo, lo);
    const double u   = p - floor(p);                     // exact
    const double m   = u * TWO_PI_HI;
    double me        = fma(u, TWO_PI_HI, -m);
    me               = fma(u, TWO_PI_LO, me);
    me               = fma(lo, TWO_PI_HI, me);
    const double M   = m + t.phi0;                       // two-sum
    const double bb  = M - m;
    const double Mlo = ((m - (M - bb)) + (t.phi0 - bb)) + me;

    if (ell) {
        double s1, c1;
        sincos(M, &s1, &c1);
        const double two_c = 2.0 * c1;
        double cp = 1.0, sp = 0.0, ck = c1, sk = s1;                     // (cos, sin) of (k-1) M and k M
        double sumC = ell->c[0] * c1, sumS = ell->s[0] * s1;             // sum C_k cos kM, sum S_k sin kM
        double dC = -ell->c[0] * s1, dS = ell->s[0] * c1;                // their derivatives with respect to M
#pragma unroll
        for (int k = 2; k <= 7; ++k) {
            const double cn = fma(two_c, ck, -cp), sn = fma(two_c, sk, -sp);
            cp = ck; sp = sk; ck = cn; sk = sn;
            const double Ck = ell->c[k - 1], Sk = ell->s[k - 1];
            sumC = fma(Ck, cn, sumC); sumS = fma(Sk, sn, sumS);
            dC = fma(-(double)k * Ck, sn, dC); dS = fma((double)k * Sk, cn, dS);
        }
        const double dv = fma(t.A, dC, t.B * dS);                        // d(delay)/dM
        val   = fma(dv, Mlo, fma(t.A, sumC, fma(t.B, sumS, -t.d0)));
        slope = dv * t.w;
        return;
    }
    double sE, cE, r;
    if (t.circular) {
        sincos(M, &sE, &cE);
        r = 1.0;
    } else {
        const double e = t.ecc;
        double sM, cM;
        sincos(M, &sM, &cM);
        double E = M + e * sM;
        sE = sM; cE = cM;
        for (int it = 0; it < 60; ++it) {
            sincos(E, &sE, &cE);
            const double f  = (E - M) - e * sE;
            const double dE = f / (1.0 - e * cE);
            E -= dE;
            if (fabs(dE) < 1e-8) {                       // last step: second-order update, no sincos
                const double h2 = 0.5 * dE * dE;
                const double s2 = sE - dE * cE - h2 * sE;
                const double c2 = cE + dE * sE - h2 * cE;
                sE = s2; cE = c2;
                break;
            }
        }
        r = 1.0 / (1.0 - e * cE);
    }
    // first-order correction for the low part of M
    const double dE = Mlo * r;
    const double s1 = fma(dE, cE, sE);
    const double c1 = fma(-dE, sE, cE);
    val   = fma(t.A, c1, fma(t.B, s1, -t.d0));
    slope = (t.B * c1 - t.A * s1) * r * t.w;
}

// floor(x) for |x| < 2^31 through the 2^52+2^51 magic constant and a round-down add: one DADD on
// the fp64 pipe instead of a quarter-rate F2I conversion.
__device__ __forceinline__ int floor_to_int(double x)
{
    return __double2loint(__dadd_rd(x, 6755399441055744.0));
}

// ---------------------------------------------------------------------------------------------
// K1  resampler (a2 + a3).  One CTA = one tile of RS_TILE output samples of one template.
//   phase 1: exact (value, slope) knots every h samples             (fp64, sincos / Newton)
//   phase 2: cubic Hermite coefficients per segment in shared memory
//   phase 3: delta_j from 3 DFMA, s = floor(delta + 1/2), idx = j - s, gather x[idx] (read-only
//            path; the series is shared by all templates and L2-resident), 128-bit store.
//   h is chosen per template on the host so that the interpolation error is < 2e-11 samples
//   (DESIGN.md 6.1); h = 1 degenerates to the exact formula at every sample.
//   Grid is flattened: blockIdx.x = tile * n_tmpl + template, so CTAs that run together read
//   the same stretch of the series.
// ---------------------------------------------------------------------------------------------
template <bool DEBUG_IDX>
__global__ void __launch_bounds__(RS_THREADS)
k_resample(const float* __restrict__ x, float* __restrict__ y, const TmplDev* __restrict__ tmpl,
           int n_tmpl, int n, int tile, float fill, long long* __restrict__ idx_out, const EllCoef* __restrict__ ell)
{
    __shared__ double s_val[RS_MAXSEG + 1];
    __shared__ double s_slp[RS_MAXSEG + 1];
    __shared__ __align__(16) double s_coef[RS_MAXSEG][4];
    __shared__ __align__(16) float4 s_cf[RS_MAXSEG];     // fp32 copy of the cubic, relative to s_ci.x
    __shared__ int2 s_ci[RS_MAXSEG];                     // (nearest integer to the first delta, tie margin bits)

    const int b     = blockIdx.x % n_tmpl;
    const int tbase = (blockIdx.x / n_tmpl) * tile;
    const TmplDev t = tmpl[b];
    const int log2h = t.log2h;
    const int h     = 1 << log2h;
    const double inv_h = 1.0 / (double)h;
    const int sub   = min(tile, RS_MAXSEG << log2h);
    float* __restrict__ yrow = y + (size_t)b * (size_t)n;

    for (int jsub = tbase; jsub < tbase + tile; jsub += sub) {
        const int nseg = sub >> log2h;
        if (jsub != tbase) __syncthreads();
        for (int k = threadIdx.x; k <= nseg; k += RS_THREADS) {
            double v, d;
            delay_knot(t, jsub + (k << log2h), v, d, ell ? ell + b : nullptr);
            s_val[k] = v;
            s_slp[k] = d * (double)h;
        }
        __syncthreads();
        for (int k = threadIdx.x; k < nseg; k += RS_THREADS) {
            const double v0 = s_val[k], v1 = s_val[k + 1], d0 = s_slp[k], d1 = s_slp[k + 1];
            const double dv = v1 - v0;
            s_coef[k][0] = v0 + 0.5;                         // +1/2: rounding becomes a floor
            s_coef[k][1] = d0;
            s_coef[k][2] = 3.0 * dv - (2.0 * d0 + d1);
            s_coef[k][3] = (d0 + d1) - 2.0 * dv;
            const double i0 = rint(v0);
            s_cf[k] = make_float4((float)(v0 - i0), (float)d0, (float)s_coef[k][2], (float)s_coef[k][3]);
            s_ci[k] = make_int2((int)i0, __float_as_int((float)((fabs(d0) + fabs(s_coef[k][2]) + fabs(s_coef[k][3]) + 2.0) * 1e-6)));
        }
        __syncthreads();

        for (int g = threadIdx.x; g < (sub >> 2); g += RS_THREADS) {
            const int o = g << 2;
            const int j = jsub + o;
            int src[4];
            if (log2h >= 2) {
                // fp32 cubic relative to the segment's integer offset; a sample whose rounding
                // residual is within the margin of a tie is re-decided with the fp64 cubic, so the
                // integer decision is the fp64 one everywhere (3 FFMA instead of 3 DFMA per sample)
                const int seg = o >> log2h;
                const float4 f = s_cf[seg];
                const int2 ie = s_ci[seg];
                const float lim = 0.5f - __int_as_float(ie.y);
                const float inv_hf = (float)inv_h;
                float tf = (float)(o & (h - 1)) * inv_hf;
                const int jb = j - ie.x + 0x4B400000;
                bool tie = false;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float yv = fmaf(fmaf(fmaf(f.w, tf, f.z), tf, f.y), tf, f.x);
                    const float z = yv + 12582912.0f;            // 1.5 * 2^23: nearest integer in the low bits
                    src[q] = jb + q - __float_as_int(z);
                    tie |= fabsf(yv - (z - 12582912.0f)) > lim;
                    tf += inv_hf;
                }
                if (tie) {
                    const double2 c01 = *reinterpret_cast<const double2*>(&s_coef[seg][0]);
                    const double2 c23 = *reinterpret_cast<const double2*>(&s_coef[seg][2]);
                    double tt = (double)(o & (h - 1)) * inv_h;
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const double d = fma(fma(fma(c23.y, tt, c23.x), tt, c01.y), tt, c01.x);
                        src[q] = j + q - floor_to_int(d);
                        tt += inv_h;
                    }
                }
            } else {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int oq  = o + q;
                    const int seg = oq >> log2h;
                    const double tt = (double)(oq & (h - 1)) * inv_h;
                    const double d = fma(fma(fma(s_coef[seg][3], tt, s_coef[seg][2]), tt, s_coef[seg][1]), tt,
                                         s_coef[seg][0]);
                    src[q] = j + q - floor_to_int(d);
                }
            }
            float4 v;
            v.x = ((unsigned)src[0] < (unsigned)n) ? __ldg(x + src[0]) : fill;
            v.y = ((unsigned)src[1] < (unsigned)n) ? __ldg(x + src[1]) : fill;
            v.z = ((unsigned)src[2] < (unsigned)n) ? __ldg(x + src[2]) : fill;
            v.w = ((unsigned)src[3] < (unsigned)n) ? __ldg(x + src[3]) : fill;
            *reinterpret_cast<float4*>(yrow + j) = v;
            if (DEBUG_IDX) {
#pragma unroll
                for (int q = 0; q < 4; ++q) idx_out[(size_t)b * (size_t)n + j + q] = (long long)src[q];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// K2  spectrum former + block median + normalisation (a5 + a6 + a7).
//   One warp = one median block of W bins.  A CTA has SP_WARPS + 1 warps on SP_WARPS + 1
//   consecutive blocks B0 .. B0 + SP_WARPS and writes the SP_WARPS * W normalised bins between the
//   centres of its first and last block (the baseline of a bin is interpolated between the two
//   block centres that enclose it): warp 0 writes the second half of its block, the last warp the
//   first half, the others their whole block.  The boundary block is therefore formed twice (by
//   two CTAs, 1/SP_WARPS extra work) instead of being exchanged through global memory.
//   Each lane keeps W/32 powers in registers, P_k = max(|X_k|^2, 1/2 |X_k - X_{k-1}|^2) with
//   X_0 <- 0 (G12-G14).  Exact block median (mean of the two middle order statistics, G15) by
//   bracket-and-select, exact bisection fallback.  After one block barrier the powers are
//   normalised in registers, P^_k = P_k ln2 / m(k), m(k) interpolated linearly between block
//   centres bW + (W-1)/2, flat outside (G15), P^_0 = 0, m <= 0 -> 0, and written once as float4:
//   the raw powers never reach HBM (RAW = true writes them too, parity tap).
//   UNPACK = true: the input is Z, the length-N/2 complex FFT of z_j = y_2j + i y_2j+1 (row
//   stride ld = N/2), and the real-series spectrum is formed on the fly,
//       2 X_k = (Z_k + conj Z_{M-k}) - i W_N^k (Z_k - conj Z_{M-k}),
//   with W_N^k = twb[block] * twn[k - block start] (two small tables made on the host in
//   extended precision).  The factor 2 is carried through the median (powers are 4x) and only
//   removed where a raw power or a median is written: it cancels in P^.
//   UNPACK = false: the input is the cuFFT R2C output (row stride ld, padded to 16 bytes).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 r2c_unpack2(float2 zk, float2 zm, float2 w)     // 2 X_k
{
    const float er = zk.x + zm.x, ei = zk.y - zm.y;
    const float orr = zk.y + zm.y, oi = zm.x - zk.x;
    return make_float2(fmaf(w.x, orr, fmaf(-w.y, oi, er)), fmaf(w.x, oi, fmaf(w.y, orr, ei)));
}

// exact order statistics W/2-1 and W/2 of the W non-negative floats held by a warp (VPT per
// lane); returns their mean.  cand = this warp's shared scratch of med_scratch_floats<W>() floats.
template <int W> __host__ __device__ constexpr int med_slots() { return (W / 32 >= 16) ? 12 : W / 32; }
template <int W> __host__ __device__ constexpr int med_scratch_floats() { return 32 * med_slots<W>(); }

// the two middle values among the bracket candidates of a warp (lane l keeps `mine` <= CK of them
// at cp[32 q]): bisection in key space (non-negative floats order like their bit patterns) on
// [L, H) until exactly one candidate (or one key) is left around rank r1
template <int CK>
__device__ __forceinline__ void median_select(const float* __restrict__ cp, int mine, int r1, int nmid, uint32_t L,
                                              uint32_t H, uint32_t& lower, uint32_t& upper)
{
    uint32_t ck[CK];
#pragma unroll
    for (int q = 0; q < CK; ++q) ck[q] = (q < mine) ? __float_as_uint(cp[32 * q]) : 0xffffffffu;
    int cl = 0, ch = nmid;                               // candidates below L, below H
    while (ch - cl > 1 && H - L > 1u) {
        const uint32_t mid = L + ((H - L) >> 1);
        int cc[3] = {0, 0, 0};                           // three short chains instead of one long one
#pragma unroll
        for (int q = 0; q < CK; ++q) cc[q % 3] += (ck[q] < mid) ? 1 : 0;
        const int c = __reduce_add_sync(0xffffffffu, cc[0] + cc[1] + cc[2]);
        if (c <= r1) { L = mid; cl = c; } else { H = mid; ch = c; }
    }
    uint32_t v1 = 0xffffffffu;
#pragma unroll
    for (int q = 0; q < CK; ++q) v1 = min(v1, ck[q] >= L ? ck[q] : 0xffffffffu);
    v1 = __reduce_min_sync(0xffffffffu, v1);             // the candidate of rank r1
    int le = 0;
    uint32_t nxt = 0xffffffffu;
#pragma unroll
    for (int q = 0; q < CK; ++q) {
        le += (ck[q] <= v1) ? 1 : 0;
        nxt = min(nxt, ck[q] > v1 ? ck[q] : 0xffffffffu);
    }
    le  = __reduce_add_sync(0xffffffffu, le);
    nxt = __reduce_min_sync(0xffffffffu, nxt);
    lower = v1;
    upper = (le >= r1 + 2) ? v1 : nxt;
}

// GUARD = false: the scratch holds W floats (a lane may keep all of its W/32 values), so the
// bracket pass needs no capacity check.
template <int W, bool GUARD = true>
__device__ __forceinline__ float warp_median(const float (&p)[W / 32], float* cand, int lane,
                                             unsigned long long* __restrict__ fallbacks)
{
    constexpr int VPT = W / 32;
    constexpr int K1 = W / 2 - 1;
    constexpr int CPL = med_slots<W>();                  // bracket values a lane can take into the selection
    // Fast path: the median of noise-like powers sits near 0.78 x the block mean, so count the
    // values below lo = 0.66 mean and keep those in [lo, hi = 0.90 mean) (about 13 % of the block,
    // 4 per lane) in a private per-lane list in shared memory (slot q of lane l at cand[l + 32 q]:
    // no scan, no compaction, no bank conflicts), then select among them.  If the two middle ranks
    // are not both inside the bracket, or a lane holds more than CPL bracket values, fall back to
    // the bisection over all W values.  The bracket test works on the bit patterns (one unsigned
    // range check per value).
    float sum = 0.f;
#pragma unroll
    for (int v = 0; v < VPT; ++v) sum += p[v];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    const float lo = sum * (0.66f / (float)W), hi = sum * (0.90f / (float)W);
    const uint32_t klo = __float_as_uint(lo), kspan = __float_as_uint(hi) - klo;
    int below = 0;
    float* __restrict__ cp = cand + lane;
    float* cw = cp;                                      // next free slot of this lane's list
#pragma unroll
    for (int v = 0; v < VPT; ++v) {
        const uint32_t k = __float_as_uint(p[v]);
        below += (k < klo) ? 1 : 0;
        if (k - klo < kspan && (!GUARD || cw < cp + 32 * CPL)) { *cw = p[v]; cw += 32; }
    }
    const int mine = (int)(cw - cp) >> 5;
    below = __reduce_add_sync(0xffffffffu, below);
    const int nmid = __reduce_add_sync(0xffffffffu, mine);
    const int most = __reduce_max_sync(0xffffffffu, mine);
    uint32_t lower, upper;
    if (below <= K1 && below + nmid >= K1 + 2 && most <= ((GUARD && CPL < VPT) ? CPL - 1 : CPL)) {
        __syncwarp();
        const int r1 = K1 - below;                       // rank among the candidates
        if (CPL > 8 && most <= 8) median_select<(CPL > 8 ? 8 : CPL)>(cp, mine, r1, nmid, klo, klo + kspan, lower, upper);
        else                      median_select<CPL>(cp, mine, r1, nmid, klo, klo + kspan, lower, upper);
        __syncwarp();
    } else {
        if (lane == 0 && fallbacks) atomicAdd(fallbacks, 1ull);
        uint32_t key[VPT];
#pragma unroll
        for (int v = 0; v < VPT; ++v) key[v] = __float_as_uint(p[v]);
        uint32_t prefix = 0;
        for (int bit = 30; bit >= 0; --bit) {
            const uint32_t cnd = prefix | (1u << bit);
            int c = 0;
#pragma unroll
            for (int v = 0; v < VPT; ++v) c += (key[v] < cnd) ? 1 : 0;
            c = __reduce_add_sync(0xffffffffu, c);
            if (c <= K1) prefix = cnd;                   // the K1-th smallest is >= cnd
        }
        int le = 0;
        uint32_t nxt = 0xffffffffu;
#pragma unroll
        for (int v = 0; v < VPT; ++v) {
            le += (key[v] <= prefix) ? 1 : 0;
            if (key[v] > prefix) nxt = min(nxt, key[v]);
        }
        le  = __reduce_add_sync(0xffffffffu, le);
        nxt = __reduce_min_sync(0xffffffffu, nxt);
        lower = prefix;
        upper = (le >= W / 2 + 1) ? prefix : nxt;
    }
    return 0.5f * (__uint_as_float(lower) + __uint_as_float(upper));
}

//   WHITE = true (plan option whiten, reading G25): the series was whitened once, the block medians
//   are skipped and P^_k = kappa P_k with the plan's constant kappa (med[] receives ln2 / kappa).
//   OVER = true (plan option interbin_oversample, reading G12b): the output is the 2x-oversampled
//   spectrum of 2 nb_in half bins, P'_2k = |X_k|^2, P'_2k+1 = (pi/4)^2 |X_k - X_k+1|^2 (X_nb = the
//   Nyquist bin of the R2C output); `nb` is then the number of half bins and a block of W half bins
//   covers W/2 input bins.
template <int W, bool UNPACK, bool RAW, bool WHITE = false, bool OVER = false>
__global__ void __launch_bounds__((SP_WARPS + 1) * 32)
k_spectrum_median(const float2* __restrict__ X, size_t ld, float* __restrict__ P, float* __restrict__ med,
                  int nb, int nblk_per_row, int cta_per_row, const float2* __restrict__ twn,
                  const float2* __restrict__ twb, unsigned long long* __restrict__ fallbacks,
                  float* __restrict__ Praw, float kappa)
{
    constexpr int VPT  = W / 32;        // powers per lane
    constexpr int ITER = W / 128;       // 4 consecutive bins per lane per iteration
    constexpr int CAP  = med_scratch_floats<W>();
    constexpr float SCALE = UNPACK ? 0.25f : 1.0f;       // powers are held as 4 P_k on the unpack path
    __shared__ float s_cand[SP_WARPS + 1][CAP];
    __shared__ float s_med[SP_WARPS + 1];
    const int row  = blockIdx.x / cta_per_row;
    const int wid  = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int blk  = (blockIdx.x % cta_per_row) * SP_WARPS + wid;     // warp SP_WARPS: the next CTA's first block
    const bool active = blk < nblk_per_row;
    const bool owner = active && wid < SP_WARPS;                      // writes the median and the raw powers

    const float2* __restrict__ Xr = X + (size_t)row * ld;
    const int base = blk * W;

    float p[VPT];
    float m_cur = 0.f;
    if (active) {
        float2 carry = make_float2(0.f, 0.f);            // X_{k-1} for lane 0 (X_{-1} = 0)
        float2 wbase = make_float2(1.f, 0.f);
        if (UNPACK) {
            wbase = __ldg(twb + blk);                    // W_N^base, N = 2 nb
            if (base > 0 && lane == 0) {
                const float2 wp = __ldg(twb + blk - 1), wl = __ldg(twn + W - 1);
                carry = r2c_unpack2(__ldg(Xr + base - 1), __ldg(Xr + (nb - base + 1)),
                                    make_float2(wp.x * wl.x - wp.y * wl.y, wp.x * wl.y + wp.y * wl.x));
            }
        } else if constexpr (!OVER) {                    // OVER counts `base` in half bins: Xr + base - 1 would lie past the row
            if (base > 0 && lane == 0) carry = __ldg(Xr + base - 1);
        }
        if constexpr (OVER) {
            static_assert(!UNPACK && !WHITE, "the oversampled spectrum is formed from the library R2C output");
            constexpr float C = 0.61685027506808491368f;     // (pi/4)^2
#pragma unroll
            for (int i = 0; i < ITER; ++i) {
                const int q0 = base + i * 128 + lane * 4;    // first of the lane's 4 half bins; input bins k0, k0+1 (+ k0+2)
                const int k0 = q0 >> 1;
                float4 a = __ldg(reinterpret_cast<const float4*>(Xr + k0));
                const float2 nx = __ldg(Xr + k0 + 2);
                if (k0 == 0) { a.x = 0.f; a.y = 0.f; }       // X_0 <- 0 before differencing (G13)
                float dx, dy;
                float4 o;
                o.x = a.x * a.x + a.y * a.y;
                dx = a.x - a.z;  dy = a.y - a.w;  o.y = C * (dx * dx + dy * dy);
                o.z = a.z * a.z + a.w * a.w;
                dx = a.z - nx.x; dy = a.w - nx.y; o.w = C * (dx * dx + dy * dy);
                if (RAW && owner) *reinterpret_cast<float4*>(Praw + (size_t)row * (size_t)nb + q0) = o;
                p[4 * i + 0] = o.x; p[4 * i + 1] = o.y; p[4 * i + 2] = o.z; p[4 * i + 3] = o.w;
            }
        } else
#pragma unroll
        for (int i = 0; i < ITER; ++i) {
            const int k0 = base + i * 128 + lane * 4;
            if (i + 2 < ITER) {                          // pull the lines of iteration i+2 into L2 (no registers held)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(Xr + k0 + 256));
                if (UNPACK) asm volatile("prefetch.global.L2 [%0];" ::"l"(Xr + (nb - k0 - 256) - 3));
            }
            float4 a = __ldg(reinterpret_cast<const float4*>(Xr + k0));
            float4 c = __ldg(reinterpret_cast<const float4*>(Xr + k0 + 2));
            if (UNPACK) {
                const float2* zm = Xr + (nb - k0);       // Z_{M-k0}; bins k0+q mirror at zm[-q]
                const float2 m0 = __ldg(k0 == 0 ? Xr : zm), m1 = __ldg(zm - 1), m2 = __ldg(zm - 2), m3 = __ldg(zm - 3);
                const float4 t01 = __ldg(reinterpret_cast<const float4*>(twn + (k0 - base)));
                const float4 t23 = __ldg(reinterpret_cast<const float4*>(twn + (k0 - base) + 2));
                const float2 x0 = r2c_unpack2(make_float2(a.x, a.y), m0, make_float2(wbase.x * t01.x - wbase.y * t01.y, wbase.x * t01.y + wbase.y * t01.x));
                const float2 x1 = r2c_unpack2(make_float2(a.z, a.w), m1, make_float2(wbase.x * t01.z - wbase.y * t01.w, wbase.x * t01.w + wbase.y * t01.z));
                const float2 x2 = r2c_unpack2(make_float2(c.x, c.y), m2, make_float2(wbase.x * t23.x - wbase.y * t23.y, wbase.x * t23.y + wbase.y * t23.x));
                const float2 x3 = r2c_unpack2(make_float2(c.z, c.w), m3, make_float2(wbase.x * t23.z - wbase.y * t23.w, wbase.x * t23.w + wbase.y * t23.z));
                a = make_float4(x0.x, x0.y, x1.x, x1.y);
                c = make_float4(x2.x, x2.y, x3.x, x3.y);
            }
            if (k0 == 0) { a.x = 0.f; a.y = 0.f; }       // X_0 <- 0 before differencing (G13)
            float px = __shfl_up_sync(0xffffffffu, c.z, 1);
            float py = __shfl_up_sync(0xffffffffu, c.w, 1);
            if (lane == 0) { px = carry.x; py = carry.y; }
            const float nx = __shfl_sync(0xffffffffu, c.z, 31);
            const float ny = __shfl_sync(0xffffffffu, c.w, 31);
            carry = make_float2(nx, ny);
            float dx, dy;
            float4 o;
            dx = a.x - px;  dy = a.y - py;  o.x = fmaxf(a.x * a.x + a.y * a.y, 0.5f * (dx * dx + dy * dy));
            dx = a.z - a.x; dy = a.w - a.y; o.y = fmaxf(a.z * a.z + a.w * a.w, 0.5f * (dx * dx + dy * dy));
            dx = c.x - a.z; dy = c.y - a.w; o.z = fmaxf(c.x * c.x + c.y * c.y, 0.5f * (dx * dx + dy * dy));
            dx = c.z - c.x; dy = c.w - c.y; o.w = fmaxf(c.z * c.z + c.w * c.w, 0.5f * (dx * dx + dy * dy));
            if (RAW && owner)
                *reinterpret_cast<float4*>(Praw + (size_t)row * (size_t)nb + k0) = make_float4(SCALE * o.x, SCALE * o.y, SCALE * o.z, SCALE * o.w);
            p[4 * i + 0] = o.x; p[4 * i + 1] = o.y; p[4 * i + 2] = o.z; p[4 * i + 3] = o.w;
        }
        if (WHITE) {                                     // constant normalisation: the owner warp writes its whole block
            if (owner) {
                float* __restrict__ Pw = P + (size_t)row * (size_t)nb + base;
#pragma unroll
                for (int i = 0; i < ITER; ++i) {
                    const int e0 = i * 128 + lane * 4;
                    float4 o = make_float4(p[4 * i] * (SCALE * kappa), p[4 * i + 1] * (SCALE * kappa), p[4 * i + 2] * (SCALE * kappa), p[4 * i + 3] * (SCALE * kappa));
                    if (base + e0 == 0) o.x = 0.f;           // P^_0 = 0
                    *reinterpret_cast<float4*>(Pw + e0) = o;
                }
                if (lane == 0) med[(size_t)row * nblk_per_row + blk] = 0.69314718055994530942f / kappa;
            }
            return;
        }
        m_cur = warp_median<W>(p, s_cand[wid], lane, owner ? fallbacks : nullptr);
        if (lane == 0) {
            s_med[wid] = m_cur;
            if (owner) med[(size_t)row * nblk_per_row + blk] = SCALE * m_cur;
        }
    }
    if (WHITE) return;
    __syncthreads();
    if (!active) return;
    // first half of the block: between the previous centre and this one; second half: this and the next
    const bool can_first  = wid > 0 || blk == 0;
    const bool can_second = wid < SP_WARPS;
    const float m_prev = (wid > 0) ? s_med[wid - 1] : m_cur;                                  // flat below the first centre
    const float m_next = (wid < SP_WARPS && blk + 1 < nblk_per_row) ? s_med[wid + 1] : m_cur; // flat above the last centre
    float* __restrict__ Pr = P + (size_t)row * (size_t)nb;
    constexpr float LN2 = 0.69314718055994530942f;
    constexpr float INV_W = 1.0f / (float)W;
#pragma unroll
    for (int i = 0; i < ITER; ++i) {
        const int e0 = i * 128 + lane * 4;               // offset of the 4 bins inside the block
        const bool second = e0 >= W / 2;
        if (!(second ? can_second : can_first)) continue;
        const float ma = second ? m_cur : m_prev, mb = second ? m_next : m_cur;
        const float f0 = ((float)(second ? e0 - W / 2 : e0 + W / 2) + 0.5f) * INV_W;
        const float st = (mb - ma) * INV_W;              // baseline step per bin
        const float b0 = fmaf(f0, mb - ma, ma);          // baseline at the first of the 4 bins
        const float b2 = fmaf(2.0f, st, b0);
        float4 o;
        if (b0 > 0.f && b2 + st > 0.f && fminf(ma, mb) > 0.f) {
            // two reciprocals per four bins; the odd bins use 1/(m + st) = (1/m)(1 - st/m) + O((st/m)^2),
            // st/m < 2^-10 |mb - ma| / m: relative error < 1e-6 for baseline ratios up to 2
            const float r0 = __fdividef(LN2, b0), r2 = __fdividef(LN2, b2);
            const float r1 = r0 * (1.0f - st * r0 * (1.0f / LN2)), r3 = r2 * (1.0f - st * r2 * (1.0f / LN2));
            o = make_float4(p[4 * i] * r0, p[4 * i + 1] * r1, p[4 * i + 2] * r2, p[4 * i + 3] * r3);
        } else {
            float* ov = reinterpret_cast<float*>(&o);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float m = fmaf((float)q, st, b0);
                ov[q] = (m > 0.f) ? __fdividef(p[4 * i + q] * LN2, m) : 0.f;
            }
        }
        if (base + e0 == 0) o.x = 0.f;                   // P^_0 = 0
        *reinterpret_cast<float4*>(Pr + base + e0) = o;
    }
}

// ---------------------------------------------------------------------------------------------
// K2t  spectrum former for the hand-written FFT (a5 + a6 + a7), input = the TRANSPOSED complex
//   spectrum Zt[k1][k2] of z_j = y_2j + i y_2j+1 (tb_fft.cuh; bin k = k1 + M1 k2, M = M1 M2 = N/2).
//   The real-series spectrum is formed on the fly (R2C unpack),
//       2 X_k = (Z_k + conj Z_{M-k}) - i W_N^k (Z_k - conj Z_{M-k}),   W_N^k = twa[k1] * twb[k2],
//   and the SAME pair (Z_k, Z_{M-k}) also gives X_{M-k} (W_N^{M-k} = -conj W_N^k), so one CTA
//   serves two mirrored tiles of 9 median blocks each and every element of Zt is read once:
//       low  tile: bins [kL0, kL0 + 9W),  kL0 = 8 g W           (blocks 8g .. 8g+8)
//       high tile: bins [hH0, hH0 + 9W),  hH0 = M - kL0 - 9W    (blocks nblk-8g-9 .. nblk-8g-1)
//   for g < nblk/16.  A tile is 9 W/M1 columns k2 of every row k1: runs of 18 complex values
//   (144 bytes) at W = 1024, M1 = 512.  Thread (k2, chunk of W/32 consecutive k1) walks k
//   upwards keeping X_{k-1} and X_{M-k+1} in registers, so each step yields the interbinned
//   powers P_k and P_{M-k+1} (G12-G14); they go to shared memory in bin order (rows of M1 + 1
//   floats: conflict-free for the transposing store and the block-order load).  Then, per side,
//   warp w takes block w of the tile into registers, selects the exact median (warp_median, its
//   own block's shared memory as scratch), and after one barrier normalises between block
//   centres exactly like k_spectrum_median and writes 8 W bins with coalesced stores.
//   Powers are carried as 4 P_k (the 1/2 of the unpack is skipped); the factor cancels in P^.
// ---------------------------------------------------------------------------------------------
constexpr int ST_MINB = 3;             // CTAs per SM the spectrum former's register budget is set for (W <= 1024)
constexpr int ST_UN = 8;               // row steps per load group of the spectrum former
constexpr int ST_WARPS = 9;
constexpr int ST_THREADS = ST_WARPS * 32;

// floats per tile in shared memory: 9 W/M1 rows of M1 + 1 floats; the high tile is stored from
// float 3 on, shifted down by two bins (see phase 1), so it needs 4 more
__host__ __device__ constexpr int st_side_floats(int W, int log2m1) { return 9 * W + 9 * (W >> log2m1) + 4; }
__host__ __device__ constexpr size_t st_smem_bytes(int W, int log2m1) { return (size_t)2 * st_side_floats(W, log2m1) * sizeof(float); }

// 2 X_k and 2 X_{M-k} from Z_k, Z_{M-k} and w = W_N^k:  E = Z_k + conj Z_{M-k}, D = Z_k - conj Z_{M-k},
// 2 X_k = E - i w D,  2 X_{M-k} = conj E - i w' D',  w' = -conj w,  D' = -conj D
__device__ __forceinline__ void st_unpack2(float2 zk, float2 zm, float2 w, float2& xk, float2& xm)
{
    const float er = zk.x + zm.x, ei = zk.y - zm.y;
    const float dx = zk.x - zm.x, dy = zk.y + zm.y;
    const float A = fmaf(w.x, dy, w.y * dx);
    const float B = fmaf(w.y, dy, -w.x * dx);
    xk = make_float2(er + A, ei + B);
    xm = make_float2(er - A, B - ei);
}

// one-off version with its own loads, for the steps just outside a thread's run; wb = W_N^{M1 k2}
template <int LOG2M1>
__device__ __forceinline__ void st_unpack_at(const float2* __restrict__ Zr, int k1, int k2, int log2m2,
                                             const float2* __restrict__ twa, float2 wb, float2& xk, float2& xm)
{
    constexpr int M1 = 1 << LOG2M1;
    const int m2 = 1 << log2m2;
    const int mr = k1 ? M1 - k1 : 0;
    const int mc = k1 ? m2 - 1 - k2 : ((m2 - k2) & (m2 - 1));          // k = 0: Z_M = Z_0
    const float2 zk = __ldg(Zr + ((size_t)k1 << log2m2) + k2);
    const float2 zm = __ldg(Zr + ((size_t)mr << log2m2) + mc);
    const float2 wa = __ldg(twa + k1);
    st_unpack2(zk, zm, make_float2(wa.x * wb.x - wa.y * wb.y, wa.x * wb.y + wa.y * wb.x), xk, xm);
    if ((k1 | k2) == 0) xk = make_float2(0.f, 0.f);                     // X_0 <- 0 before differencing (G13)
}

__device__ __forceinline__ float st_interbin(float2 x, float2 prev)
{
    const float dx = x.x - prev.x, dy = x.y - prev.y;
    return fmaxf(fmaf(x.y, x.y, x.x * x.x), 0.5f * fmaf(dy, dy, dx * dx));
}

//   WHITE = true (plan option whiten, reading G25): no medians; P^_k = kappa P_k, med[] = ln2 / kappa.
template <int W, int LOG2M1, bool RAW, bool WHITE = false>
__global__ void __launch_bounds__(ST_THREADS, (W <= 1024) ? ST_MINB : 1)
k_spectrum_t(const float2* __restrict__ Zt, float* __restrict__ P, float* __restrict__ med, int log2m2,
             int nblk, const float2* __restrict__ twa, const float2* __restrict__ twb, float2 rot,
             unsigned long long* __restrict__ fallbacks, float* __restrict__ Praw, int pf_dist, float kappa)
{
    static_assert(W >= (1 << LOG2M1), "a median block is a whole number of columns");
    constexpr int M1 = 1 << LOG2M1;
    constexpr int VPT = W / 32;
    constexpr int LC = W / 32;                           // consecutive k1 per thread
    constexpr int Q = W >> LOG2M1;                       // columns k2 per median block
    constexpr int NK2 = 9 * Q;
    constexpr int SIDE = st_side_floats(W, LOG2M1);
    extern __shared__ __align__(16) float st_sm[];
    __shared__ float s_med[2][ST_WARPS];
    float* __restrict__ s_lo = st_sm;
    float* __restrict__ s_hi = st_sm + SIDE + 3;         // bin hH0 + eh lives at s_hi[(eh - 2) + ((eh - 2) >> LOG2M1)]
    const int groups = nblk >> 4;
    const int row = blockIdx.x / groups, g = blockIdx.x % groups;
    const size_t m = (size_t)M1 << log2m2;               // bins per template
    const float2* __restrict__ Zr = Zt + (size_t)row * m;
    const int a = 8 * g * Q;                             // first column of the low tile
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // Pull the two tiles of the CTA that will take over this CTA's slot (pf_dist blocks ahead) into
    // L2: one 128-byte line per row and side (the 16-byte tail of a run is the next group's line),
    // so that DRAM keeps streaming while the resident CTAs select medians.
    if (pf_dist > 0 && blockIdx.x + pf_dist < gridDim.x) {
        const unsigned nb = blockIdx.x + pf_dist;
        const float2* __restrict__ Zn = Zt + (size_t)(nb / groups) * m;
        const int an = 8 * (int)(nb % groups) * Q;
        const size_t m2n = (size_t)1 << log2m2;
        for (int k1 = threadIdx.x; k1 < M1; k1 += ST_THREADS) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(Zn + (size_t)k1 * m2n + an));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(Zn + (size_t)k1 * m2n + (m2n - an - 8 * Q)));
        }
    }

    if constexpr (Q % 2 == 0) {
        // ---- phase 1, two columns per thread: 128-bit loads (half as many entries in the load queue the
        // kernel throttles on for the same bytes in flight).  Thread (column pair cp, row group) walks LR rows of
        // the columns k2, k2 + 1 (k2 even); their mirrors are the columns m2 - 1 - k2, m2 - 2 - k2: one aligned
        // 128-bit load too.  Two chains X_{k-1} -> X_k per thread instead of one.
        constexpr int NP = NK2 / 2, NRG = ST_THREADS / NP, LR = M1 / NRG, UN = 4;
        static_assert(NP * NRG == ST_THREADS && LR * NRG == M1 && LR % UN == 0, "pair mapping of the spectrum former");
        const int k2off = 2 * (threadIdx.x % NP), k1s = (threadIdx.x / NP) * LR;
        const int k2 = a + k2off;
        const size_t m2 = (size_t)1 << log2m2;
        const float2 wb[2] = {__ldg(twb + k2), __ldg(twb + k2 + 1)};
        float2 pl[2], ph[2];                             // 2 X_{k-1}, 2 X_{M-k+1} of the step before the run, per column
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int kk2 = k2 + j;
            const bool first = (k1s | kk2) == 0;
            const int pk1 = k1s > 0 ? k1s - 1 : M1 - 1;
            const int pk2 = k1s > 0 ? kk2 : (first ? 0 : kk2 - 1);
            st_unpack_at<LOG2M1>(Zr, pk1, pk2, log2m2, twa, k1s > 0 ? wb[j] : __ldg(twb + pk2), pl[j], ph[j]);
            if (first) { pl[j] = make_float2(0.f, 0.f); ph[j] = make_float2(0.f, 0.f); }
        }
        float* __restrict__ lo = s_lo + k1s + k2off * (M1 + 1);                           // column j: + j (M1 + 1)
        float* __restrict__ hi = s_hi + (M1 - 1 - k1s) + (9 * Q - 1 - k2off) * (M1 + 1);  // column j: - j (M1 + 1)
        const float4* zkp = reinterpret_cast<const float4*>(Zr + (size_t)k1s * m2 + k2);                      // walks down the rows
        const float4* zmp = reinterpret_cast<const float4*>(Zr + (size_t)(M1 - k1s) * m2 + (m2 - 2 - k2));   // walks up; .xy mirrors column k2 + 1, .zw column k2
        const size_t step4 = m2 >> 1;
        const float2* __restrict__ wap = twa + k1s;
#pragma unroll 1
        for (int i0 = 0; i0 < LR; i0 += UN) {
            float4 zk[UN], zm[UN];
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                zk[u] = __ldg(zkp);
                if (i0 + u == 0 && k1s == 0) {           // k1 = 0 mirrors inside row 0: columns (m2 - k2) mod m2 and m2 - k2 - 1
                    const float2 m0 = __ldg(Zr + ((m2 - k2) & (m2 - 1))), m1 = __ldg(Zr + (m2 - k2 - 1));
                    zm[u] = make_float4(m1.x, m1.y, m0.x, m0.y);
                } else zm[u] = __ldg(zmp);
                zkp += step4; zmp -= step4;
            }
            const float2 wa = __ldg(wap + i0);
            float2 w0 = make_float2(wa.x * wb[0].x - wa.y * wb[0].y, wa.x * wb[0].y + wa.y * wb[0].x);
            float2 w1 = make_float2(wa.x * wb[1].x - wa.y * wb[1].y, wa.x * wb[1].y + wa.y * wb[1].x);
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                const int it = i0 + u;
                float2 xk, xm;
                st_unpack2(make_float2(zk[u].x, zk[u].y), make_float2(zm[u].z, zm[u].w), w0, xk, xm);
                if (it == 0 && (k1s | k2) == 0) xk = make_float2(0.f, 0.f);                   // X_0 <- 0 (G13)
                lo[it] = st_interbin(xk, pl[0]);
                hi[-it] = st_interbin(ph[0], xm);
                pl[0] = xk; ph[0] = xm;
                st_unpack2(make_float2(zk[u].z, zk[u].w), make_float2(zm[u].x, zm[u].y), w1, xk, xm);
                lo[it + (M1 + 1)] = st_interbin(xk, pl[1]);
                hi[-it - (M1 + 1)] = st_interbin(ph[1], xm);
                pl[1] = xk; ph[1] = xm;
                w0 = make_float2(w0.x * rot.x - w0.y * rot.y, w0.x * rot.y + w0.y * rot.x);
                w1 = make_float2(w1.x * rot.x - w1.y * rot.y, w1.x * rot.y + w1.y * rot.x);
            }
        }
    } else {   // ---- phase 1: unpack + interbin, powers to shared memory in bin order ----
        const int k2off = threadIdx.x % NK2, k1s = (threadIdx.x / NK2) * LC;
        const int k2 = a + k2off;
        const size_t m2 = (size_t)1 << log2m2;
        const float2 wb = __ldg(twb + k2);
        // 2 X_{k-1} and 2 X_{M-k+1} of the step before the run (zero before bin 0); the loads are
        // unconditional so that they are issued together with the first group of the run
        float2 pl, ph;
        {
            const bool first = (k1s | k2) == 0;
            const int pk1 = k1s > 0 ? k1s - 1 : M1 - 1;
            const int pk2 = k1s > 0 ? k2 : (first ? 0 : k2 - 1);
            st_unpack_at<LOG2M1>(Zr, pk1, pk2, log2m2, twa, k1s > 0 ? wb : __ldg(twb + pk2), pl, ph);
            if (first) { pl = make_float2(0.f, 0.f); ph = make_float2(0.f, 0.f); }
        }
        // low bin e = k - kL0 = k1 + M1 k2off at s_lo[e + k2off]; the same step yields the high bin
        // eh = 9W + 1 - e, and eh - 2 = (M1 - 1 - k1) + M1 (9Q - 1 - k2off): both addresses move by
        // one float per step (steps e = 0, 1 land in two unused floats at the top of the high tile)
        float* __restrict__ lo = s_lo + k1s + k2off * (M1 + 1);
        float* __restrict__ hi = s_hi + (M1 - 1 - k1s) + (9 * Q - 1 - k2off) * (M1 + 1);
        const float2* zkp = Zr + (size_t)k1s * m2 + k2;                                   // walks down the rows
        const float2* zmp = Zr + (size_t)(M1 - k1s) * m2 + (m2 - 1 - k2);                 // walks up; row M1 is never read (k1s = 0 below)
        const float2* __restrict__ wap = twa + k1s;
        constexpr int UN = (LC % ST_UN == 0) ? ST_UN : 4;
#pragma unroll 1
        for (int i0 = 0; i0 < LC; i0 += UN) {
            float2 zk[UN], zm[UN];
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                zk[u] = __ldg(zkp);
                zm[u] = __ldg((i0 + u == 0 && k1s == 0) ? Zr + ((m2 - k2) & (m2 - 1)) : zmp);   // k1 = 0 mirrors inside row 0
                zkp += m2; zmp -= m2;
            }
            // W_N^k = W_N^{k1} W_N^{M1 k2}: exact table value at the head of the group, then rotated
            // by rot = W_N^1 (UN - 1 fp32 rotations: relative error below 1e-6)
            const float2 wa = __ldg(wap + i0);
            float2 w = make_float2(wa.x * wb.x - wa.y * wb.y, wa.x * wb.y + wa.y * wb.x);
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                const int it = i0 + u;
                float2 xk, xm;
                st_unpack2(zk[u], zm[u], w, xk, xm);
                if (it == 0 && (k1s | k2) == 0) xk = make_float2(0.f, 0.f);                   // X_0 <- 0 (G13)
                lo[it] = st_interbin(xk, pl);
                hi[-it] = st_interbin(ph, xm);
                pl = xk; ph = xm;
                w = make_float2(w.x * rot.x - w.y * rot.y, w.x * rot.y + w.y * rot.x);
            }
        }
    }
    if (threadIdx.x < 2) {                               // the two steps above the low tile: high bins hH0 + 1, hH0
        const int kc2 = a + NK2;                         // k = kL0 + 9W + t = (k1 = t, k2 = a + 9Q)
        const float2 wc = __ldg(twb + kc2);
        float2 x0, h0, x1, h1;
        if (threadIdx.x == 0) st_unpack_at<LOG2M1>(Zr, M1 - 1, kc2 - 1, log2m2, twa, __ldg(twb + kc2 - 1), x0, h0);
        else                  st_unpack_at<LOG2M1>(Zr, 0, kc2, log2m2, twa, wc, x0, h0);
        st_unpack_at<LOG2M1>(Zr, (int)threadIdx.x, kc2, log2m2, twa, wc, x1, h1);
        s_hi[-2 - (int)threadIdx.x] = st_interbin(h0, h1);               // eh = 1 - t: (eh - 2) + ((eh - 2) >> LOG2M1)
    }
    __syncthreads();

    constexpr float LN2 = 0.69314718055994530942f;
    constexpr float INV_W = 1.0f / (float)W;
    const bool last_pair = g == groups - 1;
#pragma unroll 1
    for (int side = 0; side < 2; ++side) {
        const int blk = side ? nblk - 8 * g - 9 + wid : 8 * g + wid;
        const bool owner = side ? wid > 0 : wid < ST_WARPS - 1;      // writes the median (and the raw powers)
        // block `wid` of the tile: bins wid W + i 32 + lane, row (wid Q + (i 32 + lane) / M1) of the tile
        float* __restrict__ sb = (side ? s_hi - 2 - (lane < 2 ? 1 : 0) : s_lo) + wid * (W + Q) + lane;
        float p[VPT];
#pragma unroll
        for (int i = 0; i < VPT; ++i) {
            // high tile: bin eh sits at (eh - 2) + ((eh - 2) >> LOG2M1); eh - 2 falls into the previous row
            // only for the first two bins of a row, i.e. lanes 0, 1 of the steps with 32 i a multiple of M1
            const int pad = (32 * i) >> LOG2M1;
            if (side && (32 * i) % M1 != 0) p[i] = sb[32 * i + pad + ((lane < 2) ? 1 : 0)];
            else                            p[i] = sb[32 * i + pad];
        }
        __syncwarp();
        if (RAW && owner) {
#pragma unroll
            for (int i = 0; i < VPT; ++i) Praw[(size_t)row * m + (size_t)blk * W + i * 32 + lane] = 0.25f * p[i];
        }
        if (WHITE) {                                     // constant normalisation: every owner warp writes its whole block
            if (owner) {
                float* __restrict__ Pw = P + (size_t)row * m + (size_t)blk * W + lane;
                const float kq = 0.25f * kappa;          // powers are carried as 4 P
#pragma unroll
                for (int i = 0; i < VPT; ++i) Pw[32 * i] = (i == 0 && blk == 0 && lane == 0) ? 0.f : p[i] * kq;
                if (lane == 0) med[(size_t)row * nblk + blk] = 0.69314718055994530942f / kappa;
            }
            continue;
        }
        // scratch for the bracket list: floats of this warp's own block (all of them are in registers now)
        const float m_cur = warp_median<W, false>(p, (side ? s_hi - 3 : s_lo) + wid * (W + Q), lane, owner ? fallbacks : nullptr);
        if (lane == 0) {
            s_med[side][wid] = m_cur;
            if (owner) med[(size_t)row * nblk + blk] = 0.25f * m_cur;
        }
        __syncthreads();
        // first half of the block: between the previous centre and this one; second half: this and the next
        bool can_first = wid > 0 || blk == 0;
        bool can_second = wid < ST_WARPS - 1 || blk == nblk - 1;
        if (side && last_pair) {                         // [centre(nblk/2-1), centre(nblk/2)) belongs to the low tile
            if (wid == 0) can_second = false;
            if (wid == 1) can_first = false;
        }
        const float m_prev = (wid > 0) ? s_med[side][wid - 1] : m_cur;              // flat below the first centre
        const float m_next = (wid < ST_WARPS - 1) ? s_med[side][wid + 1] : m_cur;   // flat above the last centre
        float* __restrict__ Pr = P + (size_t)row * m + (size_t)blk * W + lane;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (!(h ? can_second : can_first)) continue;
            const float ma = h ? m_cur : m_prev, mb = h ? m_next : m_cur;
            // baseline at bin offset eo: ma + ((eo -+ W/2) + 1/2)/W (mb - ma) = b0 + i * st32; the
            // factor 1/ln2 is folded into the baseline so that P^ = P * rcp(baseline / ln2)
            constexpr float INV_LN2 = 1.0f / LN2;
            const float st32 = (32.0f * INV_W * INV_LN2) * (mb - ma);
            const float b0 = fmaf(((float)(lane + (h ? 0 : W / 2)) + 0.5f) * INV_W, mb - ma, ma) * INV_LN2;
            if (fminf(ma, mb) > 0.f) {                   // the interpolated baseline lies between ma and mb: positive
#pragma unroll
                for (int ii = 0; ii < VPT / 2; ++ii) {
                    const int i = h * (VPT / 2) + ii;
                    float r;
                    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(fmaf((float)ii, st32, b0)));
                    float o = p[i] * r;
                    if (i == 0 && blk == 0 && lane == 0) o = 0.f;    // P^_0 = 0
                    Pr[32 * i] = o;
                }
            } else {
#pragma unroll
                for (int ii = 0; ii < VPT / 2; ++ii) {
                    const int i = h * (VPT / 2) + ii;
                    const float bl = fmaf((float)ii, st32, b0);
                    float o = (bl > 0.f) ? __fdividef(p[i], bl) : 0.f;
                    if (i == 0 && blk == 0 && lane == 0) o = 0.f;    // P^_0 = 0
                    Pr[32 * i] = o;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// K4  harmonic sum + threshold + compaction (a8 + a9).
//   S_L[k] = sum_{m=1}^{2^L} P^[(k m + 2^(L-1)) >> L]  (eq 9; G16), nested:
//   S_L = S_{L-1} + the odd-m terms.  A bin/fold over threshold becomes a candidate; the warp
//   ballots its hits and takes one atomic per warp on the device cursor (L660 "peak detection",
//   G19).  The cursor keeps counting past the capacity so that overflow is reported, not hidden.
// ---------------------------------------------------------------------------------------------
//   TAP = true (parity tap tb_debug_hsums): every S_L[k] is also written to tap[L * nb + k].
template <bool TAP>
__global__ void __launch_bounds__(256)
k_hsum_threshold(const float* __restrict__ Ph, int nb, int cta_per_row, FoldParams fp, const TmplDev* __restrict__ tmpl,
                 Candidate* __restrict__ out, unsigned long long* __restrict__ cursor,
                 unsigned long long capacity, float* __restrict__ tap)
{
    const int row = blockIdx.x / cta_per_row;
    const int k   = (blockIdx.x % cta_per_row) * 256 + threadIdx.x;
    const float* __restrict__ p = Ph + (size_t)row * (size_t)nb;
    const unsigned lane = threadIdx.x & 31;

    float S[5];
    const bool live = k < nb;
    if (live) {
        const uint32_t uk = (uint32_t)k;
        S[0] = __ldg(p + uk);
        S[1] = S[0] + __ldg(p + ((uk + 1u) >> 1));
        S[2] = S[1] + __ldg(p + ((uk + 2u) >> 2)) + __ldg(p + ((3u * uk + 2u) >> 2));
        float s = S[2];
#pragma unroll
        for (uint32_t m = 1; m < 8; m += 2) s += __ldg(p + ((m * uk + 4u) >> 3));
        S[3] = s;
#pragma unroll
        for (uint32_t m = 1; m < 16; m += 2) s += __ldg(p + ((m * uk + 8u) >> 4));
        S[4] = s;
        if (TAP) {
#pragma unroll
            for (int L = 0; L < 5; ++L) tap[(size_t)L * nb + k] = S[L];
        }
    }
    bool any = false;
    if (live) {
#pragma unroll
        for (int L = 0; L < 5; ++L) any |= (S[L] >= fp.thr[L]) && ((uint32_t)k >= fp.lo[L]);
    }
    if (__ballot_sync(0xffffffffu, any) == 0u) return;
#pragma unroll
    for (int L = 0; L < 5; ++L) {
        const bool hit = live && (S[L] >= fp.thr[L]) && ((uint32_t)k >= fp.lo[L]);
        const unsigned mask = __ballot_sync(0xffffffffu, hit);
        if (mask == 0u) continue;
        unsigned long long basepos = 0;
        if (lane == (unsigned)(__ffs(mask) - 1)) basepos = atomicAdd(cursor, (unsigned long long)__popc(mask));
        basepos = __shfl_sync(0xffffffffu, basepos, __ffs(mask) - 1);
        if (hit) {
            const unsigned long long pos = basepos + (unsigned long long)__popc(mask & ((1u << lane) - 1u));
            if (pos < capacity) {
                Candidate c;
                c.template_id = __ldg(&tmpl[row].id);
                c.fold = (uint32_t)L;
                c.bin = (uint32_t)k;
                c.power = S[L];
                c.sigma = (sqrtf(S[L]) - fp.mu[L]) * fp.inv_s[L];
                c.pad = 0u;
                out[pos] = c;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// K4t  tiled harmonic summer (a8 + a9) for Nb >= HS_T.  Same sums as k_hsum_threshold.
//   One CTA = HS_T consecutive top-harmonic bins of one template; a pair of threads = 16
//   consecutive bins k = k0 + 16 q + r (one thread r < 8, the other r >= 8).  For harmonic m/2^L (odd m) those 16 bins read the m*(16>>L)+1
//   consecutive values starting at (m k0 >> L) + m q (16>>L), and WHICH of them bin r takes,
//   (m r + 2^(L-1)) >> L, is a compile-time constant: after unrolling there is no index
//   arithmetic left, 9.4 loads per bin instead of 16, and every add is register-to-register.
//   The 14 regions (m/4, m/8, m/16) of the normalised spectrum are staged in shared memory by
//   TMA 1-D bulk copies (cp.async.bulk + mbarrier: no load/store instructions spent on staging);
//   lane strides m*(16>>L) words with 32/64/128-bit accesses are bank-conflict free for odd m.
//   Folds 0 and 1 come straight from global memory with coalesced 128-bit loads.
//   Templates are processed row-major so that one template's spectrum (2N bytes) stays in L2
//   while its 8.5 reads per bin are served (L2 -> SM traffic 17N bytes per template).
// ---------------------------------------------------------------------------------------------
constexpr int HS_T = 2048;
constexpr int HS_THREADS = HS_T / 8;

__host__ __device__ constexpr int hs_len(int L, int m) { return m * (HS_T >> L) + 4; }
__host__ __device__ constexpr int hs_off(int L, int m)
{
    int o = 0;
    for (int l = 2; l <= 4; ++l)
        for (int mm = 1; mm < (1 << l); mm += 2) {
            if (l == L && mm == m) return o;
            o += hs_len(l, mm);
        }
    return o;
}
constexpr int HS_SMEM_FLOATS = hs_off(5, 1);

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// One thread = 8 consecutive bins k = k0 + 16 q + 8 HALF + r, r < 8 (HALF is uniform per warp, so
// a warp's lanes keep the conflict-free stride of m*(16>>L) words).  With r' = r + 8 HALF the
// value bin r takes from the staged span of group q is (M r' + 2^(L-1)) >> L, a compile-time
// constant; the thread loads only the NV values its 8 bins touch, starting OFF words into the span.
template <int L, int M, int HALF>
__device__ __forceinline__ void hs_accumulate(const float* __restrict__ sm, int q, float (&acc)[8])
{
    constexpr int STEP = M * (16 >> L);              // words between consecutive groups' spans
    constexpr int RND = 1 << (L - 1);
    constexpr bool VEC2 = (STEP % 2 == 0);           // even lane stride: 64-bit loads (32-bit ones would be 2-way bank conflicts)
    constexpr int OFF0 = (M * 8 * HALF + RND) >> L;  // first value the 8 bins touch
    constexpr int OFF = VEC2 ? (OFF0 & ~1) : OFF0;
    constexpr int NV = ((M * (7 + 8 * HALF) + RND) >> L) - OFF + 1;
    const float* sp = sm + hs_off(L, M) + q * STEP + OFF;
    float v[NV + 1];
    if constexpr (VEC2) {                            // the regions carry 4 floats of padding
#pragma unroll
        for (int i = 0; i < NV; i += 2) {
            const float2 t = *reinterpret_cast<const float2*>(sp + i);
            v[i] = t.x; v[i + 1] = t.y;
        }
    } else {
#pragma unroll
        for (int i = 0; i < NV; ++i) v[i] = sp[i];
    }
#pragma unroll
    for (int r = 0; r < 8; ++r) acc[r] += v[((M * (r + 8 * HALF) + RND) >> L) - OFF];
}

// rare path: emit the hits of one fold with a warp-aggregated atomic per bin offset
template <int L>
__device__ __forceinline__ void hs_emit(const float (&acc)[8], uint32_t kq, const FoldParams& fp, uint32_t tid,
                                        Candidate* __restrict__ out, unsigned long long* __restrict__ cursor,
                                        unsigned long long capacity)
{
    const unsigned lane = threadIdx.x & 31;
#pragma unroll
    for (int r = 0; r < 8; ++r) {                    // unrolled: acc[] must stay in registers
        const uint32_t k = kq + (uint32_t)r;
        const bool hit = (acc[r] >= fp.thr[L]) && (k >= fp.lo[L]);
        const unsigned mask = __ballot_sync(0xffffffffu, hit);
        if (mask == 0u) continue;
        const int leader = __ffs(mask) - 1;
        unsigned long long basepos = 0;
        if ((int)lane == leader) basepos = atomicAdd(cursor, (unsigned long long)__popc(mask));
        basepos = __shfl_sync(0xffffffffu, basepos, leader);
        if (hit) {
            const unsigned long long pos = basepos + (unsigned long long)__popc(mask & ((1u << lane) - 1u));
            if (pos < capacity) {
                Candidate c;
                c.template_id = tid; c.fold = (uint32_t)L; c.bin = k; c.power = acc[r];
                c.sigma = (sqrtf(acc[r]) - fp.mu[L]) * fp.inv_s[L];
                c.pad = 0u;
                out[pos] = c;
            }
        }
    }
}

template <int L>
__device__ __forceinline__ void hs_check(const float (&acc)[8], uint32_t kq, const FoldParams& fp, uint32_t tid,
                                         Candidate* __restrict__ out, unsigned long long* __restrict__ cursor,
                                         unsigned long long capacity)
{
    const float thr = fp.thr[L];
    const float mx = fmaxf(fmaxf(fmaxf(acc[0], acc[1]), fmaxf(acc[2], acc[3])), fmaxf(fmaxf(acc[4], acc[5]), fmaxf(acc[6], acc[7])));
    if (__any_sync(0xffffffffu, mx >= thr)) hs_emit<L>(acc, kq, fp, tid, out, cursor, capacity);
}

// issue the 14 bulk copies of one tile's regions into `sm`, completion on `bar` (one thread)
__device__ __forceinline__ void hs_stage(float* sm, const float* __restrict__ p, int k0, uint64_t* bar)
{
    mbar_expect_tx(bar, (uint32_t)(HS_SMEM_FLOATS * sizeof(float)));
#pragma unroll
    for (int L = 2; L <= 4; ++L)
#pragma unroll
        for (int m = 1; m < (1 << L); m += 2)
            bulk_g2s(sm + hs_off(L, m), p + (((size_t)m * (size_t)k0) >> L), (uint32_t)(hs_len(L, m) * sizeof(float)), bar);
}

struct HsDirect {                                    // folds 0 and 1 of one thread's 8 bins, from global memory
    float4 a0, a1, h0;
    float  h1;
};
__device__ __forceinline__ HsDirect hs_load_direct(const float* __restrict__ p, uint32_t kq)
{
    HsDirect d;
    const float4* a = reinterpret_cast<const float4*>(p + kq);
    d.a0 = __ldg(a); d.a1 = __ldg(a + 1);
    const float* h = p + (kq >> 1);                  // kq is a multiple of 8
    d.h0 = __ldg(reinterpret_cast<const float4*>(h));
    d.h1 = __ldg(h + 4);
    return d;
}

// sums + checks of one thread's 8 bins of the tile staged in `sm`
template <bool TAP>
__device__ __forceinline__ void hs_tap(const float (&acc)[8], float* __restrict__ tap)
{
    if (TAP) {
        *reinterpret_cast<float4*>(tap) = make_float4(acc[0], acc[1], acc[2], acc[3]);
        *reinterpret_cast<float4*>(tap + 4) = make_float4(acc[4], acc[5], acc[6], acc[7]);
    }
}

template <int HALF, bool TAP>
__device__ __forceinline__ void hs_tile_body(const float* __restrict__ sm, int q, const HsDirect& d, uint32_t kq,
                                             uint64_t* bar, uint32_t parity, const FoldParams& fp, uint32_t tid,
                                             Candidate* __restrict__ out, unsigned long long* __restrict__ cursor,
                                             unsigned long long capacity, float* __restrict__ tap, size_t nb)
{
    float acc[8] = {d.a0.x, d.a0.y, d.a0.z, d.a0.w, d.a1.x, d.a1.y, d.a1.z, d.a1.w};   // fold 0: the bin itself
    hs_tap<TAP>(acc, tap + kq);
    hs_check<0>(acc, kq, fp, tid, out, cursor, capacity);
    {                                                // fold 1: + P^[(k+1)>>1], 5 values from kq/2 on
        const float v[5] = {d.h0.x, d.h0.y, d.h0.z, d.h0.w, d.h1};
#pragma unroll
        for (int r = 0; r < 8; ++r) acc[r] += v[(r + 1) >> 1];
    }
    hs_tap<TAP>(acc, tap + nb + kq);
    hs_check<1>(acc, kq, fp, tid, out, cursor, capacity);

    mbar_wait(bar, parity);
    hs_accumulate<2, 1, HALF>(sm, q, acc);
    hs_accumulate<2, 3, HALF>(sm, q, acc);
    hs_tap<TAP>(acc, tap + 2 * nb + kq);
    hs_check<2>(acc, kq, fp, tid, out, cursor, capacity);
    hs_accumulate<3, 1, HALF>(sm, q, acc);
    hs_accumulate<3, 3, HALF>(sm, q, acc);
    hs_accumulate<3, 5, HALF>(sm, q, acc);
    hs_accumulate<3, 7, HALF>(sm, q, acc);
    hs_tap<TAP>(acc, tap + 3 * nb + kq);
    hs_check<3>(acc, kq, fp, tid, out, cursor, capacity);
    hs_accumulate<4, 1, HALF>(sm, q, acc);
    hs_accumulate<4, 3, HALF>(sm, q, acc);
    hs_accumulate<4, 5, HALF>(sm, q, acc);
    hs_accumulate<4, 7, HALF>(sm, q, acc);
    hs_accumulate<4, 9, HALF>(sm, q, acc);
    hs_accumulate<4, 11, HALF>(sm, q, acc);
    hs_accumulate<4, 13, HALF>(sm, q, acc);
    hs_accumulate<4, 15, HALF>(sm, q, acc);
    hs_tap<TAP>(acc, tap + 4 * nb + kq);
    hs_check<4>(acc, kq, fp, tid, out, cursor, capacity);
}

// A CTA walks `tpc` consecutive tiles of one template with two staging buffers: while tile t is
// summed out of one buffer the bulk copies of tile t+1 land in the other, and the fold-0/1
// values of tile t+1 are already on their way to registers, so no warp waits on memory once the
// first tile is in.  Warps 0-3 take bins 0-7 of every group of 16, warps 4-7 bins 8-15: 16 warps
// per SM instead of 8 on the same staged bytes (the staging, not the registers, limits residency).
//   TAP = true (parity tap tb_debug_hsums): every S_L[k] is also written to tap[L * nb + k].
constexpr int HS_BUFS = 2;
template <bool TAP>
__global__ void __launch_bounds__(HS_THREADS, 2)
k_hsum_tile(const float* __restrict__ Ph, int nb, int groups_per_row, int tpc, FoldParams fp, const TmplDev* __restrict__ tmpl,
            Candidate* __restrict__ out, unsigned long long* __restrict__ cursor, unsigned long long capacity,
            float* __restrict__ tap)
{
    extern __shared__ __align__(16) float hs_sm[];   // two buffers of HS_SMEM_FLOATS
    __shared__ __align__(8) uint64_t bar[2];
    const int row   = blockIdx.x / groups_per_row;
    const int tile0 = (blockIdx.x % groups_per_row) * tpc;
    const float* __restrict__ p = Ph + (size_t)row * (size_t)nb;
    const uint32_t tid = __ldg(&tmpl[row].id);
    const int q = threadIdx.x & (HS_T / 16 - 1), half = threadIdx.x / (HS_T / 16);

    if (threadIdx.x == 0) { mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); }
    __syncthreads();
    if (threadIdx.x == 0) hs_stage(hs_sm, p, tile0 * HS_T, &bar[0]);
    HsDirect nxt = hs_load_direct(p, (uint32_t)(tile0 * HS_T + 16 * q + 8 * half));

    for (int t = 0; t < tpc; ++t) {
        const int k0 = (tile0 + t) * HS_T;
        const uint32_t kq = (uint32_t)(k0 + 16 * q + 8 * half);
        const float* sm = hs_sm + (t & 1) * HS_SMEM_FLOATS;
        if (t + 1 < tpc && threadIdx.x == 0)         // the other buffer was released by the barrier that ended tile t-1
            hs_stage(hs_sm + ((t + 1) & 1) * HS_SMEM_FLOATS, p, k0 + HS_T, &bar[(t + 1) & 1]);
        const HsDirect d = nxt;
        if (t + 1 < tpc) nxt = hs_load_direct(p, kq + HS_T);
        const uint32_t parity = (uint32_t)((t >> 1) & 1);
        if (half) hs_tile_body<1, TAP>(sm, q, d, kq, &bar[t & 1], parity, fp, tid, out, cursor, capacity, tap, (size_t)nb);
        else      hs_tile_body<0, TAP>(sm, q, d, kq, &bar[t & 1], parity, fp, tid, out, cursor, capacity, tap, (size_t)nb);
        __syncthreads();                             // every thread is done with buffer t&1: it may be refilled
    }
}

// fp64 partial sums of the series (fill value): block b sums the elements b*256+t, stride
// gridDim*256, per thread in index order, then the 256 threads in a fixed tree -> acc[b]
__global__ void __launch_bounds__(256) k_sum_f64(const float* __restrict__ x, size_t n, double* __restrict__ acc)
{
    __shared__ double s_w[8];
    double s = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        s += (double)x[i];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += s_w[w];
        acc[blockIdx.x] = t;
    }
}

}  // namespace tb
