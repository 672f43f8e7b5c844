// tb_fft.cuh -- hand-written two-pass (four-step) FFT of the resampled series, with the
// nearest-neighbour gather fused into the first pass's load (steps a2+a3+a4 of include/tb.h).
//
// The real series y[0..N) of one template is transformed as the complex series
// z_j = y_{2j} + i y_{2j+1}, j < M = N/2, with M = M1 * M2 ("apply the
// resampling ... and then calculate an FFT"; G11: forward, unnormalised):
//
//   j = j1*M2 + j2,  k = k1 + M1*k2
//   Z[k1 + M1 k2] = sum_{j2} W_M^{j2 k1} ( sum_{j1} z[j1 M2 + j2] W_M1^{j1 k1} ) W_M2^{j2 k2}
//
//   K0  k_delay_segments  exact (value, slope) knots of the delay every h samples -> one cubic
//                         Hermite record per segment (fp64 + an fp32 copy with a safety margin)
//   P1  k_fft_cols        per CTA a bundle of C = 16 columns j2 (M1 = 512 rows, 256 at 2^17):
//                         gathers z straight from the series in runs of 32 samples (the
//                         resampled series is never written), M1-point FFTs in shared memory,
//                         times W_M^{j2 k1}, writes T[k1][j2] in 128-byte runs   (4N bytes out)
//   P2  k_fft_rows_t      per CTA R rows k1: M2-point FFTs (M2 = 256..8192), writes the
//                         TRANSPOSED spectrum Zt[k1][k2] (bin k = k1 + M1 k2), so that both its
//                         loads and its stores are fully contiguous              (4N in, 4N out)
//   the transposition back to bin order and the R2C unpack X_k = E_k + W_N^k O_k are fused into
//   the spectrum former k_spectrum_t (below), which reads Zt in runs of >= 128 bytes.
//
// In-CTA FFT of length L = R1*256 (R1 in {1,...,32}): three in-place steps over a 3-D view
// [a < R1][b < 16][c < 16] of the data, physical index a*PA + b*PB + c (the pitches are chosen per
// kernel so that all three access patterns are bank-conflict free for 64-bit elements):
//   step 1 over a (radix R1, fused with the global load), twiddle W_L^{(16b+c) ka}
//   step 2 over b (radix 16),                              twiddle W_256^{c kb}
//   step 3 over c (radix 16, fused with the global store); output k = ka + R1 kb + 16 R1 kc.
#pragma once
#include "tb_kernels.cuh"

namespace tb {

constexpr int COLS_MINB = 3;            // CTAs per SM the pass-1 register budget is set for
constexpr int ROWS_MINB = 2;            // CTAs per SM the pass-2 register budget is set for (2 measured faster than 3)
constexpr int A0_UNROLL = 4;            // rows per batch of independent segment-record loads (x R1 points)
constexpr int A1_UNROLL = 4;            // rows per batch of independent gather loads
constexpr int FFT_PB = 17;            // pitch of the b axis (16 + 1)
constexpr int FFT_PA = 16 * FFT_PB;   // pitch of the a axis
constexpr int FFT_THREADS = 256;

struct SegRec {                       // one Hermite segment of the delay, 64 bytes
    float  f0, f1, f2, f3;            // fp32 cubic in t in [0,1): delta - i0 = f0 + t(f1 + t(f2 + t f3))
    int    i0;                        // nearest integer to the segment's first delta
    float  eps;                       // |rounding residual| beyond 0.5 - eps -> decide in fp64
    int    pad0, pad1;
    double d0, d1, d2, d3;            // fp64 cubic of delta + 1/2 (the k_resample coefficients)
};
static_assert(sizeof(SegRec) == 64, "segment record");

// Complex arithmetic on the packed fp32x2 pipe of sm_100 (FADD2 / FFMA2: one issue slot per complex
// add, three per complex multiply instead of two and four); the kernels are issue-bound, not FMA-bound.
__device__ __forceinline__ float2 cadd(float2 a, float2 b)
{
    float2 r;
    asm("{ .reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; add.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 csub(float2 a, float2 b)
{
    float2 r;
    asm("{ .reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; sub.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 cmul(float2 a, float2 w)      // (a.x, a.x) * w + (-a.y w.y, a.y w.x)
{
    float2 r;
    const float cx = -a.y * w.y, cy = a.y * w.x;
    asm("{ .reg .b64 ra, rb, rc, rd; mov.b64 ra, {%2,%2}; mov.b64 rb, {%3,%4}; mov.b64 rc, {%5,%6}; fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(w.x), "f"(w.y), "f"(cx), "f"(cy));
    return r;
}
__device__ __forceinline__ float2 mul_mi(float2 a) { return make_float2(a.y, -a.x); }   // a * (-i)

// forward 4-point DFT of (x0,x1,x2,x3), natural order in and out
__device__ __forceinline__ void fft4(float2& x0, float2& x1, float2& x2, float2& x3)
{
    const float2 t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), t3 = mul_mi(csub(x1, x3));
    x0 = cadd(t0, t2); x2 = csub(t0, t2); x1 = cadd(t1, t3); x3 = csub(t1, t3);
}

template <int R> __device__ __forceinline__ void fft_reg(float2 (&v)[R]);

template <> __device__ __forceinline__ void fft_reg<1>(float2 (&)[1]) {}
template <> __device__ __forceinline__ void fft_reg<2>(float2 (&v)[2])
{
    const float2 a = v[0], b = v[1];
    v[0] = cadd(a, b); v[1] = csub(a, b);
}
template <> __device__ __forceinline__ void fft_reg<4>(float2 (&v)[4]) { fft4(v[0], v[1], v[2], v[3]); }
template <> __device__ __forceinline__ void fft_reg<8>(float2 (&v)[8])
{
    // n = 2 n1 + n2, k = k1 + 4 k2: 4-point over n1, twiddle W8^{n2 k1}, 2-point over n2
    constexpr float H = 0.70710678118654752440f;
    fft4(v[0], v[2], v[4], v[6]);                 // n2 = 0 -> A[k1][0] in v[0],v[2],v[4],v[6]
    fft4(v[1], v[3], v[5], v[7]);                 // n2 = 1 -> A[k1][1] in v[1],v[3],v[5],v[7]
    v[3] = cmul(v[3], make_float2(H, -H));        // W8^1
    v[5] = mul_mi(v[5]);                          // W8^2
    v[7] = cmul(v[7], make_float2(-H, -H));       // W8^3
    float2 o[8];
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
        o[k1]     = cadd(v[2 * k1], v[2 * k1 + 1]);
        o[k1 + 4] = csub(v[2 * k1], v[2 * k1 + 1]);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = o[i];
}
template <> __device__ __forceinline__ void fft_reg<16>(float2 (&v)[16])
{
    // n = 4 n1 + n2, k = k1 + 4 k2: 4-point over n1, twiddle W16^{n2 k1}, 4-point over n2
    constexpr float C1 = 0.92387953251128675613f, S1 = 0.38268343236508977173f, H = 0.70710678118654752440f;
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) fft4(v[n2], v[4 + n2], v[8 + n2], v[12 + n2]);   // A[k1][n2] at v[4 k1 + n2]
    v[5]  = cmul(v[5],  make_float2(C1, -S1));    // k1=1,n2=1: W16^1
    v[6]  = cmul(v[6],  make_float2(H, -H));      // W16^2
    v[7]  = cmul(v[7],  make_float2(S1, -C1));    // W16^3
    v[9]  = cmul(v[9],  make_float2(H, -H));      // k1=2,n2=1: W16^2
    v[10] = mul_mi(v[10]);                        // W16^4
    v[11] = cmul(v[11], make_float2(-H, -H));     // W16^6
    v[13] = cmul(v[13], make_float2(S1, -C1));    // k1=3,n2=1: W16^3
    v[14] = cmul(v[14], make_float2(-H, -H));     // W16^6
    v[15] = cmul(v[15], make_float2(-C1, S1));    // W16^9
    float2 o[16];
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
        float2 a = v[4 * k1], b = v[4 * k1 + 1], c = v[4 * k1 + 2], d = v[4 * k1 + 3];
        fft4(a, b, c, d);                         // over n2 -> k2
        o[k1] = a; o[k1 + 4] = b; o[k1 + 8] = c; o[k1 + 12] = d;
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = o[i];
}

template <> __device__ __forceinline__ void fft_reg<32>(float2 (&v)[32])
{
    // decimation in frequency: u_i = v_i + v_{i+16}, d_i = (v_i - v_{i+16}) W32^i;
    // X[2k] = FFT16(u)[k], X[2k+1] = FFT16(d)[k]
    constexpr float C32[16] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                               0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                               0.19509032201612826785f, 0.0f, -0.19509032201612826785f, -0.38268343236508977173f,
                               -0.55557023301960222474f, -0.70710678118654752440f, -0.83146961230254523708f,
                               -0.92387953251128675613f, -0.98078528040323044913f};
    constexpr float S32[16] = {0.0f, 0.19509032201612826785f, 0.38268343236508977173f, 0.55557023301960222474f,
                               0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f,
                               0.98078528040323044913f, 1.0f, 0.98078528040323044913f, 0.92387953251128675613f,
                               0.83146961230254523708f, 0.70710678118654752440f, 0.55557023301960222474f,
                               0.38268343236508977173f, 0.19509032201612826785f};
    float2 u[16], d[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        u[i] = cadd(v[i], v[i + 16]);
        const float2 t = csub(v[i], v[i + 16]);
        d[i] = (i == 0) ? t : (i == 8) ? mul_mi(t) : cmul(t, make_float2(C32[i], -S32[i]));
    }
    fft_reg<16>(u);
    fft_reg<16>(d);
#pragma unroll
    for (int k = 0; k < 16; ++k) { v[2 * k] = u[k]; v[2 * k + 1] = d[k]; }
}

// step 2 of the in-CTA FFT for one slot: work item w in [0, 16 R1): (ka, c) = (w >> 4, w & 15)
template <int PA, int PB>
__device__ __forceinline__ void fft_step2(float2* __restrict__ slot, int w, const float2* __restrict__ tw2)
{
    const int c = w & 15;
    float2* p = slot + (w >> 4) * PA + c;
    float2 v[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) v[b] = p[b * PB];
    fft_reg<16>(v);
#pragma unroll
    for (int kb = 1; kb < 16; ++kb) v[kb] = cmul(v[kb], tw2[kb * 16 + c]);
#pragma unroll
    for (int kb = 0; kb < 16; ++kb) p[kb * PB] = v[kb];
}

// ---------------------------------------------------------------------------------------------
// K0  Hermite segment records of the delay for every template of the chunk.
//   One CTA = 256 consecutive segments of one template (257 exact knots, one per thread of its
//   nine warps: the 257th knot must not double the fp64 latency chain of thread 0).  Output
//   record s of template b at seg[b * seg_stride + s].  Same knots and fp64 coefficients as k_resample.
// ---------------------------------------------------------------------------------------------
constexpr int K0_THREADS = 288;
__global__ void __launch_bounds__(K0_THREADS)
k_delay_segments(const TmplDev* __restrict__ tmpl, int n_tmpl, int n, SegRec* __restrict__ seg, size_t seg_stride,
                 int cta_per_tmpl, const EllCoef* __restrict__ ell)
{
    __shared__ double s_val[257], s_slp[257];
    const int b = blockIdx.x % n_tmpl;
    const int s0 = (blockIdx.x / n_tmpl) * 256;
    const TmplDev t = tmpl[b];
    const int log2h = t.log2h;
    const int nseg = n >> log2h;
    if (s0 >= nseg) return;
    const double h = (double)(1 << log2h);
    if (threadIdx.x <= 256) {
        const int k = threadIdx.x;
        double v, d;
        delay_knot(t, (s0 + k) << log2h, v, d, ell ? ell + b : nullptr);
        s_val[k] = v; s_slp[k] = d * h;
    }
    __syncthreads();
    // records are staged piece-major in shared memory (4 pieces of 16 bytes, pitch 257) and written
    // out as one contiguous, fully coalesced stretch: direct 64-byte-strided stores left the
    // kernel waiting on the store queue (lg_throttle / drain in the ncu capture)
    __shared__ float4 s_piece[4][257];
    if (threadIdx.x < 256) {
        const double v0 = s_val[threadIdx.x], v1 = s_val[threadIdx.x + 1], g0 = s_slp[threadIdx.x], g1 = s_slp[threadIdx.x + 1];
        const double dv = v1 - v0;
        const double d0 = v0 + 0.5, d1 = g0, d2 = 3.0 * dv - (2.0 * g0 + g1), d3 = (g0 + g1) - 2.0 * dv;
        const double i0 = rint(v0);
        const float eps = (float)((fabs(d1) + fabs(d2) + fabs(d3) + 2.0) * 1e-6);
        s_piece[0][threadIdx.x] = make_float4((float)(v0 - i0), (float)d1, (float)d2, (float)d3);
        s_piece[1][threadIdx.x] = make_float4(__int_as_float((int)i0), eps, 0.f, 0.f);
        s_piece[2][threadIdx.x] = make_float4(__int_as_float(__double2loint(d0)), __int_as_float(__double2hiint(d0)),
                                              __int_as_float(__double2loint(d1)), __int_as_float(__double2hiint(d1)));
        s_piece[3][threadIdx.x] = make_float4(__int_as_float(__double2loint(d2)), __int_as_float(__double2hiint(d2)),
                                              __int_as_float(__double2loint(d3)), __int_as_float(__double2hiint(d3)));
    }
    __syncthreads();
    const int nrec = min(256, nseg - s0);
    float4* __restrict__ out = reinterpret_cast<float4*>(seg + (size_t)b * seg_stride + s0);
    for (int g = threadIdx.x; g < 4 * nrec; g += K0_THREADS) out[g] = s_piece[g & 3][g >> 2];
}

// source indices of the output sample pair (nn, nn+1), nn even (a3): fp32 cubic of the segment
// the pair lies in; a sample whose rounding residual is within eps of a tie is re-decided in
// fp64 with k_resample's coefficients, so the integer decision is the fp64 one everywhere.
__device__ __forceinline__ int2 source_pair(const SegRec* __restrict__ segs, int nn, int log2h, float inv_h)
{
    const SegRec* r = segs + (nn >> log2h);
    const float4 f = __ldg(reinterpret_cast<const float4*>(r));
    const int2 ie = __ldg(reinterpret_cast<const int2*>(r) + 2);
    const int o = nn & ((1 << log2h) - 1);
    const float t0 = (float)o * inv_h, t1 = t0 + inv_h;
    const float y0 = fmaf(fmaf(fmaf(f.w, t0, f.z), t0, f.y), t0, f.x);
    const float y1 = fmaf(fmaf(fmaf(f.w, t1, f.z), t1, f.y), t1, f.x);
    const float z0 = y0 + 12582912.0f, z1 = y1 + 12582912.0f;      // 1.5 * 2^23: round to nearest integer
    const int base = nn - ie.x + 0x4B400000;
    int2 src = make_int2(base - __float_as_int(z0), base + 1 - __float_as_int(z1));
    const float lim = 0.5f - __int_as_float(ie.y);
    const bool tie0 = fabsf(y0 - (z0 - 12582912.0f)) > lim, tie1 = fabsf(y1 - (z1 - 12582912.0f)) > lim;
    if (tie0 || tie1) {                                           // rare (about 2 eps per sample)
        const double2 c01 = __ldg(reinterpret_cast<const double2*>(r) + 2);
        const double2 c23 = __ldg(reinterpret_cast<const double2*>(r) + 3);
        const double ta = (double)o * (double)inv_h, tb = (double)(o + 1) * (double)inv_h;
        if (tie0) src.x = nn - floor_to_int(fma(fma(fma(c23.y, ta, c23.x), ta, c01.y), ta, c01.x));
        if (tie1) src.y = nn + 1 - floor_to_int(fma(fma(fma(c23.y, tb, c23.x), tb, c01.y), tb, c01.x));
    }
    return src;
}

// ---------------------------------------------------------------------------------------------
// phase A0 of pass 1: source indices of the thread's NIT * R1 points (rows j1 = a 256 + NW0 it
// relative to the thread's first row, samples nn, nn + 1), parked as int2 at
// myslot[a APITCH + it ITPITCH] (written and read back by the same thread: no barrier).
// ---------------------------------------------------------------------------------------------
// CLAMP: an out-of-range index is replaced by n, where the plan keeps the fill value (x[n]), so
// that the gather needs no bounds test (the debug taps keep the raw index).
template <bool CLAMP>
__device__ __forceinline__ int2 clamp_pair(int2 s, int n)
{
    if (CLAMP) { s.x = (int)min((unsigned)s.x, (unsigned)n); s.y = (int)min((unsigned)s.y, (unsigned)n); }
    return s;
}

template <int R1, int C, int APITCH, int ITPITCH, bool CLAMP>
__device__ __forceinline__ void cols_park_indices(const SegRec* __restrict__ segs, int log2h, float inv_h,
                                                  float2* __restrict__ myslot, int nn0, int row_shift, int n)
{
    constexpr int NW0 = FFT_THREADS / C, NIT = 256 / NW0;
    constexpr int UA0 = (A0_UNROLL * 2 / R1 > 0) ? A0_UNROLL * 2 / R1 : 1;      // 2 A0_UNROLL points per batch of loads
    if ((1 << log2h) >= 2 * C) {
        // h >= 2C: the 2C-sample run of a row lies inside one segment, the offset o of a sample in
        // its segment is the same for every row of the thread, and the record index is linear in j1
        const int o = nn0 & ((1 << log2h) - 1);
        const float t0 = (float)o * inv_h, t1 = t0 + inv_h;
        const char* __restrict__ rec0 = reinterpret_cast<const char*>(segs + (nn0 >> log2h));
        const int rec_shift = row_shift - log2h + 6;                           // log2 bytes between the records of rows j1, j1 + 1
        static_assert(NIT * R1 <= 32, "one tie flag per point of the thread");
        unsigned ties = 0;                                                     // points with a sample too close to a rounding tie for fp32
#pragma unroll UA0
        for (int it = 0; it < NIT; ++it) {
#pragma unroll
            for (int a = 0; a < R1; ++a) {
                const int j1 = a * 256 + NW0 * it;                             // row relative to w0
                const char* r = rec0 + ((unsigned)j1 << rec_shift);            // < 2^26 bytes
                const float4 f = __ldg(reinterpret_cast<const float4*>(r));
                const int2 ie = __ldg(reinterpret_cast<const int2*>(r) + 2);
                const int nn = nn0 + (j1 << row_shift);
                const float y0 = fmaf(fmaf(fmaf(f.w, t0, f.z), t0, f.y), t0, f.x);
                const float y1 = fmaf(fmaf(fmaf(f.w, t1, f.z), t1, f.y), t1, f.x);
                const float z0 = y0 + 12582912.0f, z1 = y1 + 12582912.0f;      // 1.5 * 2^23: round to nearest integer
                const int base = nn - ie.x + 0x4B400000;
                const float lim = 0.5f - __int_as_float(ie.y);
                const float res = fmaxf(fabsf(y0 - (z0 - 12582912.0f)), fabsf(y1 - (z1 - 12582912.0f)));
                ties |= (res > lim ? 1u : 0u) << (it * R1 + a);
                *reinterpret_cast<int2*>(myslot + a * APITCH + it * ITPITCH) =
                    clamp_pair<CLAMP>(make_int2(base - __float_as_int(z0), base + 1 - __float_as_int(z1)), n);
            }
        }
        while (ties) {                                                         // rare (about 2 eps per sample): decide in fp64
            const int e = __ffs(ties) - 1;
            ties &= ties - 1;
            const int a = e % R1, it = e / R1;
            const int j1 = a * 256 + NW0 * it;
            const char* r = rec0 + ((unsigned)j1 << rec_shift);
            const int nn = nn0 + (j1 << row_shift);
            const double2 c01 = __ldg(reinterpret_cast<const double2*>(r) + 2);
            const double2 c23 = __ldg(reinterpret_cast<const double2*>(r) + 3);
            const double ta = (double)o * (double)inv_h, tb = (double)(o + 1) * (double)inv_h;
            *reinterpret_cast<int2*>(myslot + a * APITCH + it * ITPITCH) =
                clamp_pair<CLAMP>(make_int2(nn - floor_to_int(fma(fma(fma(c23.y, ta, c23.x), ta, c01.y), ta, c01.x)),
                                            nn + 1 - floor_to_int(fma(fma(fma(c23.y, tb, c23.x), tb, c01.y), tb, c01.x))), n);
        }
    } else {
#pragma unroll 2
        for (int it = 0; it < NIT; ++it) {
#pragma unroll
            for (int a = 0; a < R1; ++a) {
                const int nn = nn0 + ((a * 256 + NW0 * it) << row_shift);
                *reinterpret_cast<int2*>(myslot + a * APITCH + it * ITPITCH) = clamp_pair<CLAMP>(source_pair(segs, nn, log2h, inv_h), n);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// P1  gather + column FFTs.  CTA = C columns [c0, c0+C) of template b, all M1 = R1*256 rows.
//   blockIdx.x = bundle * n_tmpl + b (template fastest: co-resident CTAs gather from the same
//   stretch of the series, which stays in L2).  A row of the CTA's tile is a run of 2C
//   consecutive output samples: with C = 16 one 128-byte stretch of the series (shifted by the
//   delay) and one segment record serve 16 threads.
// ---------------------------------------------------------------------------------------------
//   DIRECT = true: no gather.  The kernel is the middle pass of the three-pass FFT (N >= 2^25):
//   "template" b is one row of T seen as an [L][2^log2m2] matrix, transformed in place over its
//   first index with the twiddle W_m^{j2 k1}, m = L 2^log2m2 (blockIdx.x = b * bundles + bundle).
template <int R1, int C, bool DEBUG, bool DIRECT = false>
__global__ void __launch_bounds__(FFT_THREADS, COLS_MINB)
k_fft_cols(const float* __restrict__ x, const SegRec* __restrict__ seg, size_t seg_stride,
           const TmplDev* __restrict__ tmpl, int n_tmpl, int n, int log2m2, float fill,
           const float2* __restrict__ tw1, const float2* __restrict__ tw2g, float2* __restrict__ T,
           long long* __restrict__ idx_out, float* __restrict__ y_out, int pf_dist)
{
    constexpr int PB = FFT_PB, PA = FFT_PA;
    constexpr int L = R1 * 256;                    // M1
    constexpr int LP = R1 * PA + 16 / C;           // slot pitch: 16/C mod 16 keeps the column-fastest accesses conflict free
    extern __shared__ __align__(16) float2 fsm[];
    float2* tw2 = fsm + C * LP;
    const int bundles = (1 << log2m2) / C;
    const int b  = DIRECT ? blockIdx.x / bundles : blockIdx.x % n_tmpl;
    const int c0 = (DIRECT ? blockIdx.x % bundles : blockIdx.x / n_tmpl) * C;
    const size_t m = (size_t)L << log2m2;          // M
    const int log2h = DIRECT ? 0 : tmpl[b].log2h;
    const float inv_h = 1.0f / (float)(1 << log2h);
    const SegRec* __restrict__ segs = seg + (size_t)b * seg_stride;
    float2* __restrict__ Tb = T + (size_t)b * m;

    tw2[threadIdx.x] = __ldg(tw2g + threadIdx.x);
    // Pull the segment records of the CTA pf_dist blocks ahead (written by K0 just before, about
    // half of them no longer in L2) into L2: one record per row of its tile.
    if (!DEBUG && !DIRECT && pf_dist > 0 && blockIdx.x + pf_dist < gridDim.x) {
        const unsigned nb = blockIdx.x + pf_dist;
        const int bn = nb % n_tmpl, cn = (nb / n_tmpl) * C;
        const int lh = __ldg(&tmpl[bn].log2h);
        const SegRec* __restrict__ sn = seg + (size_t)bn * seg_stride;
        for (int j1 = threadIdx.x; j1 < L; j1 += FFT_THREADS)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(sn + ((int)((((size_t)j1 << log2m2) + cn) << 1) >> lh)));
    }

    // phase A0: source indices of every point of the tile, parked as an int2 in the point's own
    // shared-memory slot (written and read back by the same thread: no barrier).  Splitting the
    // index computation from the gather turns two dependent memory latencies per point
    // (segment record -> series sample) into two loops of independent loads.
    // Thread (col, w0) = (tid % C, tid / C) owns the points (a, w = w0 + NW0 it), it < NIT: row
    // j1 = a 256 + w of the tile, samples nn, nn + 1 with nn = 2 (j1 M2 + c0 + col).
    static_assert((C == 16 || C == 8) && FFT_THREADS == 256, "thread -> (col, w0) mapping");
    constexpr int NW0 = FFT_THREADS / C, NIT = 256 / NW0;                      // w0 values, steps per thread
    constexpr int UA1 = (A1_UNROLL * 2 / R1 > 0) ? A1_UNROLL * 2 / R1 : 1;
    constexpr int ITP = (NW0 / 16) * PB;                                       // slot pitch of one step
    const int col = threadIdx.x & (C - 1), w0 = threadIdx.x / C;
    float2* __restrict__ myslot = fsm + col * LP + (w0 >> 4) * PB + (w0 & 15); // + a PA + it ITP
    const int nn0 = (int)((((size_t)w0 << log2m2) + c0 + col) << 1);
    const int row_shift = log2m2 + 1;                                          // samples between rows j1, j1 + 1
    if (DIRECT && pf_dist > 0 && blockIdx.x + pf_dist < gridDim.x) {            // tile of a later CTA -> L2 (one line per row)
        const unsigned nb = blockIdx.x + pf_dist;
        const float2* __restrict__ Tn = T + (size_t)(nb / bundles) * m + (nb % bundles) * C;
        for (int j1 = threadIdx.x; j1 < L; j1 += FFT_THREADS) asm volatile("prefetch.global.L2 [%0];" ::"l"(Tn + ((size_t)j1 << log2m2)));
    }
    if (!DIRECT) cols_park_indices<R1, C, PA, ITP, !DEBUG>(segs, log2h, inv_h, myslot, nn0, row_shift, n);
    // phase A1: gather (independent loads), radix-R1 over a, twiddle, back to the same slots
#pragma unroll UA1
    for (int it = 0; it < NIT; ++it) {
        const int w = w0 + NW0 * it;
        float2* p = myslot + it * ITP;
        float2 v[R1];
#pragma unroll
        for (int a = 0; a < R1; ++a) {
            if (DIRECT) {
                v[a] = __ldcs(Tb + ((size_t)(a * 256 + w) << log2m2) + c0 + col);
                continue;
            }
            const int2 sp = *reinterpret_cast<const int2*>(p + a * PA);
            if (DEBUG) {                             // raw indices: test here; otherwise clamped to n, x[n] = fill
                v[a].x = ((unsigned)sp.x < (unsigned)n) ? __ldg(x + sp.x) : fill;
                v[a].y = ((unsigned)sp.y < (unsigned)n) ? __ldg(x + sp.y) : fill;
            } else {
                v[a].x = __ldg(x + sp.x);
                v[a].y = __ldg(x + sp.y);
            }
            if (DEBUG) {
                const size_t nn = (size_t)b * n + (size_t)(nn0 + ((a * 256 + NW0 * it) << row_shift));
                idx_out[nn] = sp.x; idx_out[nn + 1] = sp.y;
                y_out[nn] = v[a].x; y_out[nn + 1] = v[a].y;
            }
        }
        fft_reg<R1>(v);
#pragma unroll
        for (int ka = 1; ka < R1; ++ka) v[ka] = cmul(v[ka], __ldg(tw1 + ka * 256 + w));
#pragma unroll
        for (int ka = 0; ka < R1; ++ka) p[ka * PA] = v[ka];
    }
    __syncthreads();
    // phase B: radix 16 over b
    for (int i = threadIdx.x; i < 16 * R1 * C; i += FFT_THREADS) fft_step2<PA, PB>(fsm + (i / (16 * R1)) * LP, i % (16 * R1), tw2);
    __syncthreads();
    // phase C: radix 16 over c, four-step twiddle W_M^{j2 k1}, store T[k1][j2].  item: col fastest
    for (int i = threadIdx.x; i < 16 * R1 * C; i += FFT_THREADS) {
        const int col = i % C, w = i / C;          // w = ka*16 + kb
        const int ka = w >> 4, kb = w & 15;
        const float2* p = fsm + col * LP + ka * PA + kb * PB;
        float2 v[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) v[c] = p[c];
        fft_reg<16>(v);
        const int j2 = c0 + col;
        const int kbase = ka + R1 * kb;            // k1 = kbase + 16 R1 kc
        // W_M^{j2 k1} = W_M^{j2 kbase} * g^kc, g = W_M^{16 R1 j2}; both arguments are exact in fp32
        const float inv_m = 1.0f / (float)m;
        float sb, cb, sg, cg;
        sincospif(-2.0f * (float)(j2 * kbase) * inv_m, &sb, &cb);
        sincospif(-2.0f * (float)(j2 * 16 * R1) * inv_m, &sg, &cg);
        const float2 g1 = make_float2(cg, sg);
        const float2 g2 = cmul(g1, g1), g4 = cmul(g2, g2), g8 = cmul(g4, g4);
        float2 pw[16];
        pw[0] = make_float2(cb, sb);
        pw[1] = cmul(pw[0], g1);
        pw[2] = cmul(pw[0], g2); pw[3] = cmul(pw[1], g2);
#pragma unroll
        for (int q = 0; q < 4; ++q) pw[4 + q] = cmul(pw[q], g4);
#pragma unroll
        for (int q = 0; q < 8; ++q) pw[8 + q] = cmul(pw[q], g8);
        float2* out = Tb + ((size_t)kbase << log2m2) + j2;
        const unsigned kstep = (unsigned)(16 * R1) << log2m2;                  // 15 kstep < M <= 2^27 elements
#pragma unroll
        for (int kc = 0; kc < 16; ++kc) __stcs(out + (unsigned)kc * kstep, cmul(v[kc], pw[kc]));   // streamed: read once by pass 2
    }
}

// ---------------------------------------------------------------------------------------------
// P1 for M1 = 512 = 32 x 16: two in-CTA steps instead of three.  Row j1 = 16 a + c (a < 32,
// c < 16), output k1 = ka + 32 kc.  Thread (col, c) gathers its 32 rows a (the same rows, and
// the same phase A0, as in k_fft_cols<2, 16>), does the radix-32 step in registers, multiplies
// by W_512^{c ka} (table twc[ka 16 + c]) and writes slot[col][ka][c]; after ONE barrier the work
// item (col, ka) does the radix-16 step over c, the four-step twiddle W_M^{j2 k1} and the
// streaming stores of T[k1][j2].  One shared-memory round trip and one barrier less per point
// than the 2 x 16 x 16 scheme, and a pitch of 513 keeps every access conflict free.
// ---------------------------------------------------------------------------------------------
constexpr int C32_PK = 16, C32_LP = 32 * C32_PK + 1;
constexpr size_t C32_SMEM = (size_t)16 * C32_LP * sizeof(float2);

// ---------------------------------------------------------------------------------------------
// index phase of k_fft_cols32.  Work item = 4 consecutive output samples (columns 2q, 2q + 1 of row
// r): thread (q, r0) = (tid & 7, tid >> 3) takes rows r0 + 32 i, i < 16.  One segment record (two
// loads), one row address and one tie limit now serve four samples instead of two, the cubic's
// arguments t_k are the same for every row of the thread, and every h >= 4 goes through the same
// code (a group of 4 aligned samples never straddles a segment).  The indices are parked as int2 in
// the points' own slots, slot(col, r) = fsm[col LP + r]; a barrier separates this from the gather,
// which reads them with the (col, c) mapping of the FFT.
// ---------------------------------------------------------------------------------------------
template <bool CLAMP>
__device__ __forceinline__ void cols32_park_indices(const SegRec* __restrict__ segs, int log2h, float inv_h,
                                                    float2* __restrict__ fsm, int c0, int row_shift, int n)
{
    constexpr int LP = C32_LP;
    constexpr float MAGIC = 12582912.0f;                                       // 1.5 * 2^23: round to nearest integer
    const int q = threadIdx.x & 7, r0 = threadIdx.x >> 3;
    const int nnq = (c0 + 2 * q) << 1;                                         // first sample of the group in row 0
    const int o = nnq & ((1 << log2h) - 1);
    float t[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) t[k] = (float)(o + k) * inv_h;
    const int rec_shift = row_shift - log2h + 6;                               // log2 bytes between the records of rows r, r + 1
    const char* __restrict__ rec = reinterpret_cast<const char*>(segs + (nnq >> log2h)) + ((size_t)r0 << rec_shift);
    const unsigned rec_step = 32u << rec_shift;                                // rows r, r + 32; 15 rec_step < 2^27
    const int nn0 = nnq + (r0 << row_shift), nn_step = 32 << row_shift;
    int2* __restrict__ slot = reinterpret_cast<int2*>(fsm + (2 * q) * LP + r0);
    unsigned ties = 0;                                                         // items with a sample too close to a rounding tie for fp32
#pragma unroll 8
    for (int i = 0; i < 16; ++i) {
        const char* r = rec + (size_t)((unsigned)i * rec_step);
        const float4 f = __ldg(reinterpret_cast<const float4*>(r));
        const int2 ie = __ldg(reinterpret_cast<const int2*>(r) + 2);
        float y[4], z[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            y[k] = fmaf(fmaf(fmaf(f.w, t[k], f.z), t[k], f.y), t[k], f.x);
            z[k] = y[k] + MAGIC;
        }
        const float res = fmaxf(fmaxf(fabsf(y[0] - (z[0] - MAGIC)), fabsf(y[1] - (z[1] - MAGIC))),
                                fmaxf(fabsf(y[2] - (z[2] - MAGIC)), fabsf(y[3] - (z[3] - MAGIC))));
        ties |= (res > 0.5f - __int_as_float(ie.y) ? 1u : 0u) << i;
        const int base = nn0 + i * nn_step - ie.x + 0x4B400000;
        slot[i * 32]      = clamp_pair<CLAMP>(make_int2(base - __float_as_int(z[0]), base + 1 - __float_as_int(z[1])), n);
        slot[i * 32 + LP] = clamp_pair<CLAMP>(make_int2(base + 2 - __float_as_int(z[2]), base + 3 - __float_as_int(z[3])), n);
    }
    while (ties) {                                                             // rare (about 4 eps per item): decide in fp64
        const int i = __ffs(ties) - 1;
        ties &= ties - 1;
        const char* r = rec + (size_t)((unsigned)i * rec_step);
        const double2 c01 = __ldg(reinterpret_cast<const double2*>(r) + 2);
        const double2 c23 = __ldg(reinterpret_cast<const double2*>(r) + 3);
        const int nn = nn0 + i * nn_step;
        int s[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const double tk = (double)(o + k) * (double)inv_h;
            s[k] = nn + k - floor_to_int(fma(fma(fma(c23.y, tk, c23.x), tk, c01.y), tk, c01.x));
        }
        slot[i * 32]      = clamp_pair<CLAMP>(make_int2(s[0], s[1]), n);
        slot[i * 32 + LP] = clamp_pair<CLAMP>(make_int2(s[2], s[3]), n);
    }
}

//   TW = false: the four-step twiddle W_M^{j2 k1} is left to pass 2 (k_fft_rows_t<32, true>, N = 2^23): pass 1 is
//   bound by instruction issue, pass 2 by HBM with issue slots to spare.
template <bool DEBUG, bool TW = true>
__global__ void __launch_bounds__(FFT_THREADS, COLS_MINB)
k_fft_cols32(const float* __restrict__ x, const SegRec* __restrict__ seg, size_t seg_stride,
             const TmplDev* __restrict__ tmpl, int n_tmpl, int n, int log2m2, float fill,
             const float2* __restrict__ twc, float2* __restrict__ T,
             long long* __restrict__ idx_out, float* __restrict__ y_out, int pf_dist)
{
    constexpr int C = 16, PK = C32_PK, LP = C32_LP, L = 512;
    extern __shared__ __align__(16) float2 fsm[];
    const int b  = blockIdx.x % n_tmpl;
    const int c0 = (blockIdx.x / n_tmpl) * C;
    const size_t m = (size_t)L << log2m2;          // M
    const int log2h = tmpl[b].log2h;
    const float inv_h = 1.0f / (float)(1 << log2h);
    const SegRec* __restrict__ segs = seg + (size_t)b * seg_stride;
    float2* __restrict__ Tb = T + (size_t)b * m;

    if (!DEBUG && pf_dist > 0 && blockIdx.x + pf_dist < gridDim.x) {           // segment records of a later CTA -> L2
        const unsigned nb = blockIdx.x + pf_dist;
        const int bn = nb % n_tmpl, cn = (nb / n_tmpl) * C;
        const int lh = __ldg(&tmpl[bn].log2h);
        const SegRec* __restrict__ sn = seg + (size_t)bn * seg_stride;
        for (int j1 = threadIdx.x; j1 < L; j1 += FFT_THREADS)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(sn + ((int)((((size_t)j1 << log2m2) + cn) << 1) >> lh)));
    }

    const int col = threadIdx.x & 15, c = threadIdx.x >> 4;
    float2* __restrict__ myslot = fsm + col * LP + c;                          // + a' PK, a' = 16 a + it
    const int nn0 = (int)((((size_t)c << log2m2) + c0 + col) << 1);
    const int row_shift = log2m2 + 1;
    cols32_park_indices<!DEBUG>(segs, log2h, inv_h, fsm, c0, row_shift, n);
    __syncthreads();                                                           // the indices were parked by other threads
    {   // gather (64 independent loads), radix 32 over a', twiddle, back to the same slots
        float2 v[32];
#pragma unroll
        for (int a = 0; a < 32; ++a) {
            const int2 sp = *reinterpret_cast<const int2*>(myslot + a * PK);
            if (DEBUG) {                             // raw indices: test here; otherwise clamped to n, x[n] = fill
                v[a].x = ((unsigned)sp.x < (unsigned)n) ? __ldg(x + sp.x) : fill;
                v[a].y = ((unsigned)sp.y < (unsigned)n) ? __ldg(x + sp.y) : fill;
            } else {
                v[a].x = __ldg(x + sp.x);
                v[a].y = __ldg(x + sp.y);
            }
            if (DEBUG) {
                const size_t nn = (size_t)b * n + (size_t)(nn0 + ((16 * a) << row_shift));
                idx_out[nn] = sp.x; idx_out[nn + 1] = sp.y;
                y_out[nn] = v[a].x; y_out[nn + 1] = v[a].y;
            }
        }
        fft_reg<32>(v);
        myslot[0] = v[0];
        {   // W_512^{c ka} = q[ka >> 3] * t[ka & 7] from two table values (see fft_rows_body)
            float2 t[8], q[4];
            t[1] = __ldg(twc + 16 + c);
            q[1] = __ldg(twc + 8 * 16 + c);
            t[2] = cmul(t[1], t[1]); t[3] = cmul(t[2], t[1]); t[4] = cmul(t[2], t[2]);
            t[5] = cmul(t[4], t[1]); t[6] = cmul(t[4], t[2]); t[7] = cmul(t[4], t[3]);
            q[2] = cmul(q[1], q[1]); q[3] = cmul(q[2], q[1]);
#pragma unroll
            for (int ka = 1; ka < 8; ++ka) myslot[ka * PK] = cmul(v[ka], t[ka]);
#pragma unroll
            for (int h = 1; h < 4; ++h) {
                myslot[8 * h * PK] = cmul(v[8 * h], q[h]);
#pragma unroll
                for (int l = 1; l < 8; ++l) myslot[(8 * h + l) * PK] = cmul(v[8 * h + l], cmul(q[h], t[l]));
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 16 * 32; i += FFT_THREADS) {                 // item (col, ka), col fastest
        const int cl = i & 15, ka = i >> 4;
        const float2* p = fsm + cl * LP + ka * PK;
        float2 v[16];
#pragma unroll
        for (int cc = 0; cc < 16; ++cc) v[cc] = p[cc];
        fft_reg<16>(v);
        const int j2 = c0 + cl;
        if constexpr (!TW) {
            float2* out = Tb + ((size_t)ka << log2m2) + j2;
            const unsigned kstep = 32u << log2m2;
#pragma unroll
            for (int kc = 0; kc < 16; ++kc) __stcs(out + (unsigned)kc * kstep, v[kc]);
            continue;
        }
        // W_M^{j2 k1} = W_M^{j2 ka} * g^kc, g = W_M^{32 j2}; both arguments are exact in fp32
        const float inv_m = 1.0f / (float)m;
        float sb, cb, sg, cg;
        sincospif(-2.0f * (float)(j2 * ka) * inv_m, &sb, &cb);
        sincospif(-2.0f * (float)(j2 * 32) * inv_m, &sg, &cg);
        const float2 g1 = make_float2(cg, sg);
        const float2 g2 = cmul(g1, g1), g4 = cmul(g2, g2), g8 = cmul(g4, g4);
        float2 pw[16];
        pw[0] = make_float2(cb, sb);
        pw[1] = cmul(pw[0], g1);
        pw[2] = cmul(pw[0], g2); pw[3] = cmul(pw[1], g2);
#pragma unroll
        for (int q = 0; q < 4; ++q) pw[4 + q] = cmul(pw[q], g4);
#pragma unroll
        for (int q = 0; q < 8; ++q) pw[8 + q] = cmul(pw[q], g8);
        float2* out = Tb + ((size_t)ka << log2m2) + j2;
        const unsigned kstep = 32u << log2m2;
#pragma unroll
        for (int kc = 0; kc < 16; ++kc) __stcs(out + (unsigned)kc * kstep, cmul(v[kc], pw[kc]));   // streamed: read once by pass 2
    }
}

// ---------------------------------------------------------------------------------------------
// P1 for M1 = 1024 = 32 x 32 (N = 2^25): bundles of C = 8 columns (64 KB of shared memory), two radix-32
// steps in registers with one barrier between them, the index phase per 4-sample work item as in
// k_fft_cols32.  Row j1 = 32 a + c, output k1 = ka + 32 kc.  slot(col, r) = fsm[col LP + 33 (r / 32) +
// r % 32], LP = 32 * 33 + 2: the index phase, the gather (thread (col, c): rows c + 32 a), the
// write-back (ka in place of a) and the second step (thread (col, ka): 32 consecutive c) are all
// conflict free for 64-bit elements.  twc: [ka 32 + c] = W_1024^{c ka}.
// ---------------------------------------------------------------------------------------------
constexpr int C1K_LP = 32 * 33 + 2;
constexpr size_t C1K_SMEM = (size_t)8 * C1K_LP * sizeof(float2);

template <bool DEBUG>
__global__ void __launch_bounds__(FFT_THREADS, 2)        // measured: 2 CTAs/SM (128 registers) 151 us per template at 2^25, 3 CTAs (80) 174
k_fft_cols1k(const float* __restrict__ x, const SegRec* __restrict__ seg, size_t seg_stride,
             const TmplDev* __restrict__ tmpl, int n_tmpl, int n, int log2m2, float fill,
             const float2* __restrict__ twc, float2* __restrict__ T,
             long long* __restrict__ idx_out, float* __restrict__ y_out, int pf_dist)
{
    constexpr int C = 8, LP = C1K_LP, L = 1024;
    constexpr float MAGIC = 12582912.0f;
    extern __shared__ __align__(16) float2 fsm[];
    const int b  = blockIdx.x % n_tmpl;
    const int c0 = (blockIdx.x / n_tmpl) * C;
    const size_t m = (size_t)L << log2m2;          // M
    const int log2h = tmpl[b].log2h;
    const float inv_h = 1.0f / (float)(1 << log2h);
    const SegRec* __restrict__ segs = seg + (size_t)b * seg_stride;
    float2* __restrict__ Tb = T + (size_t)b * m;
    const int row_shift = log2m2 + 1;

    if (!DEBUG && pf_dist > 0 && blockIdx.x + pf_dist < gridDim.x) {           // segment records of a later CTA -> L2
        const unsigned nb = blockIdx.x + pf_dist;
        const int bn = nb % n_tmpl, cn = (nb / n_tmpl) * C;
        const int lh = __ldg(&tmpl[bn].log2h);
        const SegRec* __restrict__ sn = seg + (size_t)bn * seg_stride;
        for (int j1 = threadIdx.x; j1 < L; j1 += FFT_THREADS)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(sn + ((int)((((size_t)j1 << log2m2) + cn) << 1) >> lh)));
    }
    {   // index phase: item = 4 consecutive samples (columns 2q, 2q + 1) of row r0 + 64 i
        const int q = threadIdx.x & 3, r0 = threadIdx.x >> 2;
        const int nnq = (c0 + 2 * q) << 1;
        const int o = nnq & ((1 << log2h) - 1);
        float t[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) t[k] = (float)(o + k) * inv_h;
        const int rec_shift = row_shift - log2h + 6;
        const char* __restrict__ rec = reinterpret_cast<const char*>(segs + (nnq >> log2h)) + ((size_t)r0 << rec_shift);
        const size_t rec_step = (size_t)64 << rec_shift;
        const int nnr = nnq + (r0 << row_shift), nn_step = 64 << row_shift;
        int2* __restrict__ slot = reinterpret_cast<int2*>(fsm + (2 * q) * LP + 33 * (r0 >> 5) + (r0 & 31));   // + 66 i
        unsigned ties = 0;
#pragma unroll 8
        for (int i = 0; i < 16; ++i) {
            const char* r = rec + (size_t)i * rec_step;
            const float4 f = __ldg(reinterpret_cast<const float4*>(r));
            const int2 ie = __ldg(reinterpret_cast<const int2*>(r) + 2);
            float y[4], z[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                y[k] = fmaf(fmaf(fmaf(f.w, t[k], f.z), t[k], f.y), t[k], f.x);
                z[k] = y[k] + MAGIC;
            }
            const float res = fmaxf(fmaxf(fabsf(y[0] - (z[0] - MAGIC)), fabsf(y[1] - (z[1] - MAGIC))),
                                    fmaxf(fabsf(y[2] - (z[2] - MAGIC)), fabsf(y[3] - (z[3] - MAGIC))));
            ties |= (res > 0.5f - __int_as_float(ie.y) ? 1u : 0u) << i;
            const int base = nnr + i * nn_step - ie.x + 0x4B400000;
            slot[i * 66]      = clamp_pair<!DEBUG>(make_int2(base - __float_as_int(z[0]), base + 1 - __float_as_int(z[1])), n);
            slot[i * 66 + LP] = clamp_pair<!DEBUG>(make_int2(base + 2 - __float_as_int(z[2]), base + 3 - __float_as_int(z[3])), n);
        }
        while (ties) {                                                         // rare: decide in fp64
            const int i = __ffs(ties) - 1;
            ties &= ties - 1;
            const char* r = rec + (size_t)i * rec_step;
            const double2 c01 = __ldg(reinterpret_cast<const double2*>(r) + 2);
            const double2 c23 = __ldg(reinterpret_cast<const double2*>(r) + 3);
            const int nn = nnr + i * nn_step;
            int sidx[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double tk = (double)(o + k) * (double)inv_h;
                sidx[k] = nn + k - floor_to_int(fma(fma(fma(c23.y, tk, c23.x), tk, c01.y), tk, c01.x));
            }
            slot[i * 66]      = clamp_pair<!DEBUG>(make_int2(sidx[0], sidx[1]), n);
            slot[i * 66 + LP] = clamp_pair<!DEBUG>(make_int2(sidx[2], sidx[3]), n);
        }
    }
    __syncthreads();
    const int col = threadIdx.x & 7, c = threadIdx.x >> 3;
    {   // gather (64 independent loads), radix 32 over a, twiddle W_1024^{c ka}, back to the same slots
        float2* __restrict__ myslot = fsm + col * LP + c;                      // + 33 a
        const int nn0 = (int)((((size_t)c << log2m2) + c0 + col) << 1);
        float2 v[32];
#pragma unroll
        for (int a = 0; a < 32; ++a) {
            const int2 sp = *reinterpret_cast<const int2*>(myslot + 33 * a);
            if (DEBUG) {
                v[a].x = ((unsigned)sp.x < (unsigned)n) ? __ldg(x + sp.x) : fill;
                v[a].y = ((unsigned)sp.y < (unsigned)n) ? __ldg(x + sp.y) : fill;
                const size_t nn = (size_t)b * n + (size_t)(nn0 + ((32 * a) << row_shift));
                idx_out[nn] = sp.x; idx_out[nn + 1] = sp.y;
                y_out[nn] = v[a].x; y_out[nn + 1] = v[a].y;
            } else {
                v[a].x = __ldg(x + sp.x);
                v[a].y = __ldg(x + sp.y);
            }
        }
        fft_reg<32>(v);
        myslot[0] = v[0];
        float2 t[8], q[4];
        t[1] = __ldg(twc + 32 + c);
        q[1] = __ldg(twc + 8 * 32 + c);
        t[2] = cmul(t[1], t[1]); t[3] = cmul(t[2], t[1]); t[4] = cmul(t[2], t[2]);
        t[5] = cmul(t[4], t[1]); t[6] = cmul(t[4], t[2]); t[7] = cmul(t[4], t[3]);
        q[2] = cmul(q[1], q[1]); q[3] = cmul(q[2], q[1]);
#pragma unroll
        for (int ka = 1; ka < 8; ++ka) myslot[33 * ka] = cmul(v[ka], t[ka]);
#pragma unroll
        for (int h = 1; h < 4; ++h) {
            myslot[33 * 8 * h] = cmul(v[8 * h], q[h]);
#pragma unroll
            for (int l = 1; l < 8; ++l) myslot[33 * (8 * h + l)] = cmul(v[8 * h + l], cmul(q[h], t[l]));
        }
    }
    __syncthreads();
    {   // item (col, ka): radix 32 over c, four-step twiddle W_M^{j2 k1}, k1 = ka + 32 kc, streaming stores of T[k1][j2]
        const int ka = c;
        const float2* p = fsm + col * LP + 33 * ka;
        float2 v[32];
#pragma unroll
        for (int cc = 0; cc < 32; ++cc) v[cc] = p[cc];
        fft_reg<32>(v);
        const int j2 = c0 + col;
        const float inv_m = 1.0f / (float)m;
        float sb, cb, sg, cg;
        sincospif(-2.0f * (float)(j2 * ka) * inv_m, &sb, &cb);                 // both arguments are exact in fp32
        sincospif(-2.0f * (float)(j2 * 32) * inv_m, &sg, &cg);
        float2 t[8], bq[4];                                                    // g^l, base g^{8h}
        t[1] = make_float2(cg, sg);
        t[2] = cmul(t[1], t[1]); t[3] = cmul(t[2], t[1]); t[4] = cmul(t[2], t[2]);
        t[5] = cmul(t[4], t[1]); t[6] = cmul(t[4], t[2]); t[7] = cmul(t[4], t[3]);
        const float2 g8 = cmul(t[4], t[4]);
        bq[0] = make_float2(cb, sb);
        bq[1] = cmul(bq[0], g8); bq[2] = cmul(bq[1], g8); bq[3] = cmul(bq[2], g8);
        float2* out = Tb + ((size_t)ka << log2m2) + j2;
        const size_t kstep = (size_t)32 << log2m2;
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            __stcs(out + (size_t)(8 * h) * kstep, cmul(v[8 * h], bq[h]));
#pragma unroll
            for (int l = 1; l < 8; ++l) __stcs(out + (size_t)(8 * h + l) * kstep, cmul(v[8 * h + l], cmul(bq[h], t[l])));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// P2  row FFTs, transposed output.  CTA = R rows [k1, k1+R) of template b, row length
//   M2 = R1*256 (R1 up to 32: 8192 points, 32 values per thread in the first radix step).
//   Output Zt[k1][k2], k2 = ka + R1 kb + 16 R1 kc: the last step's work items run ka-fastest so
//   that a warp stores 32 consecutive k2 (256 bytes); the pitches PB = 16 + R1 (mod 16) and
//   PA = 16 PB + 1 keep that access, and the two before it, free of bank conflicts.
//   blockIdx.x = b * (M1/R) + row group.
// ---------------------------------------------------------------------------------------------
template <int R1> struct RowsCfg {
    static constexpr int PB = (R1 < 16) ? 16 + R1 : 17;
    static constexpr int PA = 16 * PB + 1;
    static constexpr int R = (R1 >= 8) ? 1 : 8 / R1;       // rows per CTA
    static constexpr int LP = R1 * PA;
    static constexpr int MINB = ROWS_MINB;        // CTAs per SM the register budget is set for
    static constexpr size_t SMEM = (size_t)(R * LP + 256) * sizeof(float2);
};

//   TWIN = true (R1 = 32 only): the input has not been multiplied by the four-step twiddle yet; element
//   j2 = a 256 + w of row k1 takes W_M^{j2 k1} = W_M^{k1 w} (W_M^{256 k1})^a here, from two sincospif with
//   exact arguments and a power tree, computed while the loads are in flight.
template <int R1, bool TWIN = false>
__global__ void __launch_bounds__(FFT_THREADS, RowsCfg<R1>::MINB)
k_fft_rows_t(const float2* __restrict__ T, float2* __restrict__ Zt, int log2m1, const float2* __restrict__ tw1,
             const float2* __restrict__ tw2g, int pf_dist)
{
    static_assert(!TWIN || R1 == 32, "the twiddle-on-load variant is instantiated for 8192-point rows only");
    using Cfg = RowsCfg<R1>;
    constexpr int PA = Cfg::PA, PB = Cfg::PB, R = Cfg::R, LP = Cfg::LP;
    constexpr int L = R1 * 256;                    // M2
    extern __shared__ __align__(16) float2 fsm[];
    float2* tw2 = fsm + R * LP;
    const int groups = (1 << log2m1) / R;
    const int b  = blockIdx.x / groups;
    const int k1 = (blockIdx.x % groups) * R;
    const size_t off = ((size_t)b << log2m1) * L + (size_t)k1 * L;
    const float2* __restrict__ Tb = T + off;
    float2* __restrict__ Zb = Zt + off;

    tw2[threadIdx.x] = __ldg(tw2g + threadIdx.x);
    // Pull the rows of the CTA that will take over this CTA's slot (pf_dist blocks ahead) into L2
    // with one bulk prefetch, so that DRAM keeps streaming while the resident CTAs are in their
    // compute phases (without it the reads come in bursts at CTA start and HBM idles in between).
    if (threadIdx.x == 0 && pf_dist > 0 && blockIdx.x + pf_dist < gridDim.x) {
        const float2* nxt = T + (size_t)(blockIdx.x + pf_dist) * (size_t)(R * L);
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nxt), "r"((unsigned)(R * L * sizeof(float2))) : "memory");
    }

    {   // phase A: item (r, w) = (it, threadIdx.x); every global load of the thread is issued before
        // the first butterfly so that one memory round trip covers the whole tile
        static_assert(FFT_THREADS == 256, "one work item per thread and row");
        const int w = threadIdx.x;
        float2 v[R][R1];
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int a = 0; a < R1; ++a) v[r][a] = __ldcs(Tb + (size_t)r * L + a * 256 + w);
        if constexpr (TWIN) {
            const float inv_m = 1.0f / (float)((size_t)L << log2m1);
            float sb, cb, sg, cg;
            sincospif(-2.0f * (float)(k1 * w) * inv_m, &sb, &cb);              // k1 w, 256 k1 < 2^17: exact in fp32
            sincospif(-2.0f * (float)(k1 * 256) * inv_m, &sg, &cg);
            float2 t[8], bq[4];                                                 // g^l, base g^{8h}
            t[1] = make_float2(cg, sg);
            t[2] = cmul(t[1], t[1]); t[3] = cmul(t[2], t[1]); t[4] = cmul(t[2], t[2]);
            t[5] = cmul(t[4], t[1]); t[6] = cmul(t[4], t[2]); t[7] = cmul(t[4], t[3]);
            const float2 g8 = cmul(t[4], t[4]);
            bq[0] = make_float2(cb, sb);
            bq[1] = cmul(bq[0], g8); bq[2] = cmul(bq[1], g8); bq[3] = cmul(bq[2], g8);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                v[0][8 * h] = cmul(v[0][8 * h], bq[h]);
#pragma unroll
                for (int l = 1; l < 8; ++l) v[0][8 * h + l] = cmul(v[0][8 * h + l], cmul(bq[h], t[l]));
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            fft_reg<R1>(v[r]);
            float2* p = fsm + r * LP + (w >> 4) * PB + (w & 15);
            p[0] = v[r][0];
            if constexpr (R1 == 32) {
                // W_L^{w ka} = q[ka >> 3] * t[ka & 7] from two table values (ka = 1 and 8): 29 complex
                // products on the FMA pipe instead of 29 more loads on the LSU/MIO path this kernel
                // throttles on; at most four roundings deep
                float2 t[8], q[4];
                t[1] = __ldg(tw1 + 256 + w);
                q[1] = __ldg(tw1 + 8 * 256 + w);
                t[2] = cmul(t[1], t[1]); t[3] = cmul(t[2], t[1]); t[4] = cmul(t[2], t[2]);
                t[5] = cmul(t[4], t[1]); t[6] = cmul(t[4], t[2]); t[7] = cmul(t[4], t[3]);
                q[2] = cmul(q[1], q[1]); q[3] = cmul(q[2], q[1]);
#pragma unroll
                for (int ka = 1; ka < 8; ++ka) p[ka * PA] = cmul(v[r][ka], t[ka]);
#pragma unroll
                for (int h = 1; h < 4; ++h) {
                    p[8 * h * PA] = cmul(v[r][8 * h], q[h]);
#pragma unroll
                    for (int l = 1; l < 8; ++l) p[(8 * h + l) * PA] = cmul(v[r][8 * h + l], cmul(q[h], t[l]));
                }
            } else
#pragma unroll
            for (int ka = 1; ka < R1; ++ka) p[ka * PA] = cmul(v[r][ka], __ldg(tw1 + ka * 256 + w));
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 16 * R1 * R; i += FFT_THREADS) fft_step2<PA, PB>(fsm + (i / (16 * R1)) * LP, i % (16 * R1), tw2);
    __syncthreads();
    for (int i = threadIdx.x; i < 16 * R1 * R; i += FFT_THREADS) {  // phase C: item (r, w'), ka fastest
        const int r = i / (16 * R1), wp = i % (16 * R1);
        const int ka = wp % R1, kb = wp / R1;
        const float2* p = fsm + r * LP + ka * PA + kb * PB;
        float2 v[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) v[c] = p[c];
        fft_reg<16>(v);
        float2* out = Zb + (size_t)r * L + wp;     // k2 = wp + 16 R1 kc
#pragma unroll
        for (int kc = 0; kc < 16; ++kc) __stcs(out + kc * (16 * R1), v[kc]);
    }
}

// ---------------------------------------------------------------------------------------------
// P2 for rows of M2 = 16384 points (N = 2^24 with M1 = 512): one row per CTA of 512 threads,
//   L = 32 x 512 = 32 x (16 x 32).  Thread w loads T[a 512 + w], a < 32 (all loads before the first
//   butterfly), radix 32 in registers over a, twiddle W_L^{w ka} (product tree from the table
//   values ka = 1 and 8); then per ka a 512-point FFT over w = 32 b + c in shared memory: radix 16
//   over b (items (ka, c), two per thread), twiddle W_512^{c kb}, radix 32 over c (item (ka, kb),
//   one per thread, ka fastest).  Output Zt[k1][k2], k2 = ka + 32 (kb + 16 kc): a warp stores 32
//   consecutive k2.  Element (ka, b, c) at ka PA + b PB + c with PB = 33, PA = 16 PB + 1 (odd):
//   all three access patterns are conflict free for 64-bit elements.  128 KB of shared memory:
//   one CTA per SM, so the next row is pulled into L2 while this one is transformed.
//   tw1: [w] = W_L^w, [512 + w] = W_L^{8 w};  tw512: [kb 32 + c] = W_512^{c kb}.
// ---------------------------------------------------------------------------------------------
constexpr int RW_THREADS = 512, RW_PB = 33, RW_PA = 16 * RW_PB + 1, RW_L = 16384;
constexpr size_t RW_SMEM = (size_t)(32 * RW_PA + 512) * sizeof(float2);

__global__ void __launch_bounds__(RW_THREADS, 1)
k_fft_rows_wide(const float2* __restrict__ T, float2* __restrict__ Zt, const float2* __restrict__ tw1,
                const float2* __restrict__ tw512g, int pf_dist)
{
    constexpr int PA = RW_PA, PB = RW_PB, L = RW_L;
    extern __shared__ __align__(16) float2 fsm[];
    float2* tw512 = fsm + 32 * PA;
    const float2* __restrict__ Tb = T + (size_t)blockIdx.x * L;
    float2* __restrict__ Zb = Zt + (size_t)blockIdx.x * L;
    const int w = threadIdx.x;
    tw512[w] = __ldg(tw512g + w);
    if (w == 0 && pf_dist > 0 && blockIdx.x + pf_dist < gridDim.x) {           // a later CTA's row -> L2
        const float2* nxt = T + (size_t)(blockIdx.x + pf_dist) * L;
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nxt), "r"((unsigned)(L * sizeof(float2))) : "memory");
    }
    {
        float2 v[32];
#pragma unroll
        for (int a = 0; a < 32; ++a) v[a] = __ldcs(Tb + a * 512 + w);
        fft_reg<32>(v);
        float2* p = fsm + (w >> 5) * PB + (w & 31);                            // (b, c) = (w / 32, w % 32); + ka PA
        p[0] = v[0];
        float2 t[8], q[4];
        t[1] = __ldg(tw1 + w);
        q[1] = __ldg(tw1 + 512 + w);
        t[2] = cmul(t[1], t[1]); t[3] = cmul(t[2], t[1]); t[4] = cmul(t[2], t[2]);
        t[5] = cmul(t[4], t[1]); t[6] = cmul(t[4], t[2]); t[7] = cmul(t[4], t[3]);
        q[2] = cmul(q[1], q[1]); q[3] = cmul(q[2], q[1]);
#pragma unroll
        for (int ka = 1; ka < 8; ++ka) p[ka * PA] = cmul(v[ka], t[ka]);
#pragma unroll
        for (int h = 1; h < 4; ++h) {
            p[8 * h * PA] = cmul(v[8 * h], q[h]);
#pragma unroll
            for (int l = 1; l < 8; ++l) p[(8 * h + l) * PA] = cmul(v[8 * h + l], cmul(q[h], t[l]));
        }
    }
    __syncthreads();
#pragma unroll 1
    for (int i = threadIdx.x; i < 32 * 32; i += RW_THREADS) {                  // item (ka, c): radix 16 over b
        const int c = i & 31, ka = i >> 5;
        float2* p = fsm + ka * PA + c;
        float2 v[16];
#pragma unroll
        for (int b = 0; b < 16; ++b) v[b] = p[b * PB];
        fft_reg<16>(v);
#pragma unroll
        for (int kb = 1; kb < 16; ++kb) v[kb] = cmul(v[kb], tw512[kb * 32 + c]);
#pragma unroll
        for (int kb = 0; kb < 16; ++kb) p[kb * PB] = v[kb];
    }
    __syncthreads();
    {                                                                          // item (ka, kb), ka fastest: radix 32 over c
        const int ka = threadIdx.x & 31, kb = threadIdx.x >> 5;
        const float2* p = fsm + ka * PA + kb * PB;
        float2 v[32];
#pragma unroll
        for (int c = 0; c < 32; ++c) v[c] = p[c];
        fft_reg<32>(v);
        float2* out = Zb + ka + 32 * kb;                                       // k2 = ka + 32 (kb + 16 kc)
#pragma unroll
        for (int kc = 0; kc < 32; ++kc) __stcs(out + kc * 512, v[kc]);
    }
}

// ---------------------------------------------------------------------------------------------
// Last pass of the three-pass FFT (N >= 2^25).  A row of M' = 256 * 256 points has been
// transformed over its slow index by k_fft_cols<1, 16, false, true> (U[ka][jb], twiddled); this
// kernel does the 256-point FFTs over jb for 16 consecutive ka and writes the row's spectrum in
// natural order, Zt[row][ka + 256 kb], in 128-byte runs (16 consecutive ka per kb).
//   blockIdx.x = row * 16 + group of 16 ka.
// ---------------------------------------------------------------------------------------------
constexpr int RS_ROWS = 16;
constexpr size_t RS_SMEM = (size_t)(RS_ROWS * (16 * FFT_PB + 1) + 256) * sizeof(float2);

__global__ void __launch_bounds__(FFT_THREADS, 3)
k_fft_rows_scatter(const float2* __restrict__ U, float2* __restrict__ Zt, const float2* __restrict__ tw2g, int pf_dist)
{
    constexpr int PB = FFT_PB, LP = 16 * FFT_PB + 1;
    extern __shared__ __align__(16) float2 fsm[];
    float2* tw2 = fsm + RS_ROWS * LP;
    const size_t row = blockIdx.x >> 4;
    const int ka0 = (blockIdx.x & 15) * RS_ROWS;
    const float2* __restrict__ Ub = U + (row << 16) + (size_t)ka0 * 256;
    float2* __restrict__ Zb = Zt + (row << 16) + ka0;
    tw2[threadIdx.x] = __ldg(tw2g + threadIdx.x);
    if (threadIdx.x == 0 && pf_dist > 0 && blockIdx.x + pf_dist < gridDim.x) {  // the 32 KB of a later CTA -> L2
        const float2* nxt = U + (size_t)(blockIdx.x + pf_dist) * (RS_ROWS * 256);
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nxt), "r"((unsigned)(RS_ROWS * 256 * sizeof(float2))) : "memory");
    }
    {
        const int w = threadIdx.x;                   // jb = 16 b + c
        float2 v[RS_ROWS];
#pragma unroll
        for (int r = 0; r < RS_ROWS; ++r) v[r] = __ldcs(Ub + r * 256 + w);
#pragma unroll
        for (int r = 0; r < RS_ROWS; ++r) fsm[r * LP + (w >> 4) * PB + (w & 15)] = v[r];
    }
    __syncthreads();
    fft_step2<LP, PB>(fsm + (threadIdx.x >> 4) * LP, threadIdx.x & 15, tw2);   // item (r, c): radix 16 over b
    __syncthreads();
    {
        const int r = threadIdx.x & 15, kb = threadIdx.x >> 4;                 // r fastest: 16 consecutive ka per store
        const float2* p = fsm + r * LP + kb * PB;
        float2 v[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) v[c] = p[c];
        fft_reg<16>(v);
#pragma unroll
        for (int kc = 0; kc < 16; ++kc) __stcs(Zb + (size_t)(kb + 16 * kc) * 256 + r, v[kc]);
    }
}

}  // namespace tb
