// tb_api.cu -- host side of libtb: plan, template constants (a1), chunked launch sequence,
// candidate retrieval (a10), timings and parity taps.  Boundary: include/tb.h.
#include "../../include/tb.h"
#include "tb_kernels.cuh"
#include "tb_fft.cuh"
#include "tb_reduce.cuh"
#include "tb_whiten.cuh"

#include <cufft.h>

constexpr int HS_TPC = 16;             // tiles walked by one CTA of the harmonic summer

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <map>
#include <new>
#include <set>
#include <string>
#include <deque>
#include <vector>

using namespace tb;

static_assert(sizeof(tb_candidate) == 24 && sizeof(Candidate) == 24, "candidate layout");
static_assert(sizeof(tb_template) == 40, "template layout");
static_assert(sizeof(tb_group) == 32 && sizeof(Group) == 32, "group layout");

namespace {

constexpr int N_STAGE_EVENTS = 6;   // start, delay model (K0), resample / P1, fft / P2, spectrum+median+normalise, hsum

// e[0..5] on the plan's stream; k[0], k[1] around K0 on the side stream it runs on (fused path)
struct EventSet { cudaEvent_t e[N_STAGE_EVENTS]; cudaEvent_t k[2]; bool k_used; };

}  // namespace

struct tb_plan {
    int device = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    uint64_t n = 0, nb = 0;                         // samples, FFT bins N/2
    uint64_t nsp = 0;                                // spectrum bins: nb, or 2 nb half bins with interbin_oversample (G12b)
    bool over = false;
    double tsamp = 0.0;
    uint32_t window = 1024, log2w = 10, nblk = 0;
    double f_min = 0.1;
    uint32_t k_lo = 0;
    uint64_t max_cand = 0;
    uint32_t chunk = 0;
    bool timings = false;
    bool user_fill = false, borrowed = false, l2_pinned = false;
    cudaStreamAttrValue l2_prev = {};                // access-policy window a caller-owned stream had before the plan set its own
    float fill = 0.f;
    float h_fillpad[4] = {0.f, 0.f, 0.f, 0.f};
    size_t ld = 0;                                   // complex row stride of the FFT output

    const float* d_series = nullptr;
    float* d_series_owned = nullptr;
    float* d_resampled = nullptr;                    // [chunk][n]
    float2* d_fft = nullptr;                         // [chunk][ld]
    float* d_power = nullptr;                        // [chunk][nb]
    float* d_med = nullptr;                          // [chunk][nblk]
    Candidate* d_cand = nullptr;
    unsigned long long* d_cursor = nullptr;
    TmplDev* d_tmpl = nullptr;
    size_t tmpl_cap = 0;
    TmplDev* h_tmpl = nullptr;                       // pinned staging
    size_t h_tmpl_cap = 0;
    bool ell = false;                                // delay_model 1: ELL7 series instead of the Kepler solve (f4)
    EllCoef* d_ell = nullptr;                        // [tmpl_cap], staged with the templates
    EllCoef* h_ell = nullptr;
    cudaEvent_t ev_staged = nullptr;                 // the last template upload has been consumed
    // K0 of chunk i+1 (fp64-bound, 3 % of the step) runs on a side stream under P2 / spectrum / hsum of chunk i
    cudaStream_t s_k0 = nullptr;
    cudaEvent_t ev_main = nullptr, ev_p1 = nullptr, ev_k0 = nullptr;
    bool staged_pending = false;

    // hand-written FFT path (tb_fft.cuh): M = N/2 = M1 * M2
    bool own_fft = false;
    int log2m1 = 0, log2m2 = 0;
    SegRec* d_seg = nullptr;                         // [chunk][seg_stride], grown on demand (seg_stride = n >> smallest knot spacing staged)
    size_t seg_stride = 0, seg_cap = 0;              // records per template, records allocated
    float2 *d_tw1a = nullptr, *d_tw1b = nullptr, *d_tw2 = nullptr, *d_twn = nullptr, *d_twb = nullptr, *d_twc = nullptr, *d_tw512 = nullptr;
    bool cols32 = false;                             // pass 1 as 32 x 16 (M1 = 512)
    float2 rot = {1.f, 0.f};                         // W_N^1
    int chunk_log2h = 0;                             // smallest knot spacing among the templates of the chunk being launched
    int n_sm = 148;                                  // multiprocessors of the device
    // L2 prefetch distances in CTAs (measured on B200, profiles/r01_v3.md)
    int pf_rows = 0;                                 // pass 2: two CTAs per SM ahead
    int pf_cols = 128;                               // pass 1 (segment records)
    int pf_mid = 1500, pf_scat = 1500;               // the two row passes of the three-pass FFT
    int pf_spec = 32;                                // spectrum former
    std::vector<uint32_t> order;                     // staging order of the current call: fused-path templates first
    size_t n_own = 0;                                // how many of them take the fused path

    // f2: front-end whitening once per series (tb_whiten.cuh)
    bool whiten = false, whitening_now = false;
    float kappa = 0.f;                               // P^ = kappa P for every template of a whitened series
    std::vector<uint2> zap;                          // zapped bin ranges [lo, hi)
    uint2* d_zap = nullptr;
    cufftHandle c2r_plan = 0, d2z_plan = 0;      // Z2D and D2Z of the whitening step
    bool have_c2r = false;

    std::map<uint32_t, cufftHandle> fft_plans;       // by batch size, sharing one work area
    void* d_work = nullptr;
    double* d_acc = nullptr;
    size_t work_bytes = 0;

    std::deque<EventSet> events;                   // deque: references stay valid when sets are appended
    size_t events_used = 0;
    tb_timings last = {};

    std::set<const void*> smem_ok;                   // kernels whose dynamic shared-memory limit has been raised on this device

    std::string err;
};

namespace {

int fail(tb_plan* p, int code, const std::string& msg)
{
    if (p) p->err = msg;
    return code;
}

#define TB_CUDA(p, call)                                                                               \
    do {                                                                                               \
        cudaError_t e__ = (call);                                                                      \
        if (e__ != cudaSuccess)                                                                        \
            return fail((p), e__ == cudaErrorMemoryAllocation ? TB_ERR_NOMEM : TB_ERR_CUDA,            \
                        std::string(#call) + ": " + cudaGetErrorString(e__));                          \
    } while (0)

#define TB_CUFFT(p, call)                                                                              \
    do {                                                                                               \
        cufftResult r__ = (call);                                                                      \
        if (r__ != CUFFT_SUCCESS)                                                                      \
            return fail((p), r__ == CUFFT_ALLOC_FAILED ? TB_ERR_NOMEM : TB_ERR_CUFFT,                  \
                        std::string(#call) + ": cufft error " + std::to_string((int)r__));             \
    } while (0)

// opt a kernel in to more than 48 KB of dynamic shared memory, once per plan (the attribute is per device)
int allow_smem(tb_plan* p, const void* kern, size_t bytes)
{
    if (p->smem_ok.count(kern)) return TB_OK;
    TB_CUDA(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    p->smem_ok.insert(kern);
    return TB_OK;
}

bool is_pow2(uint64_t v) { return v && !(v & (v - 1)); }
uint32_t ilog2(uint64_t v) { uint32_t l = 0; while ((1ull << (l + 1)) <= v) ++l; return l; }

// sigma map (G17): sqrt(S) for S ~ Gamma(n,1) has mean Gamma(n+1/2)/Gamma(n), variance n - mean^2
void sigma_constants(uint32_t fold, double* mu, double* s)
{
    const uint32_t n = 1u << fold;
    double m = 0.88622692545275801365;                 // Gamma(3/2)/Gamma(1) = sqrt(pi)/2
    for (uint32_t i = 1; i < n; ++i) m *= ((double)i + 0.5) / (double)i;   // Gamma(i+3/2)/Gamma(i+1)
    *mu = m;
    *s = std::sqrt((double)n - m * m);
}

// Knot spacing of the cubic Hermite interpolation of the delay: the largest
// h = 2^l <= 128 with  (h w)^4 / 384 * (tau/tsamp) * K(e) <= 2e-11 samples, where
// K(e) = R^4 + 11 e R^5 + 25 e^2 R^6 + 15 e^3 R^7, R = 1/(1-e), bounds the 4th derivative of
// A cos E + B sin E with respect to the mean anomaly.
// Appendix B of the paper: {power of e, numerator, denominator} of C_k, S_k, k = 1..7
struct EllTerm { int k, pw; double num, den; };
const EllTerm ELL_C_TERMS[] = {{1, 0, 1, 1}, {1, 2, -3, 8}, {1, 4, 5, 192}, {1, 6, -7, 9216}, {2, 1, 1, 2}, {2, 3, -1, 3}, {2, 5, 1, 16},
                               {3, 2, 3, 8}, {3, 4, -45, 128}, {3, 6, 567, 5120}, {4, 3, 1, 3}, {4, 5, -2, 5}, {5, 4, 125, 384},
                               {5, 6, -4375, 9216}, {6, 5, 27, 80}, {7, 6, 16807, 46080}};
const EllTerm ELL_S_TERMS[] = {{1, 0, 1, 1}, {1, 2, -5, 8}, {1, 4, -11, 192}, {1, 6, -457, 9216}, {2, 1, 1, 2}, {2, 3, -5, 12}, {2, 5, 1, 24},
                               {3, 2, 3, 8}, {3, 4, -51, 128}, {3, 6, 543, 5120}, {4, 3, 1, 3}, {4, 5, -13, 30}, {5, 4, 125, 384},
                               {5, 6, -4625, 9216}, {6, 5, 27, 80}, {7, 6, 16807, 46080}};

void ell_coefficients(double ecc, long double (&C)[8], long double (&S)[8])      // C[k], S[k], k = 1..7
{
    for (int k = 0; k < 8; ++k) C[k] = S[k] = 0.0L;
    for (const EllTerm& t : ELL_C_TERMS) C[t.k] += (long double)t.num / (long double)t.den * powl((long double)ecc, t.pw);
    for (const EllTerm& t : ELL_S_TERMS) S[t.k] += (long double)t.num / (long double)t.den * powl((long double)ecc, t.pw);
}

int knot_log2(double tau_over_tsamp, double w, double e, bool ell = false)
{
    const double R = 1.0 / (1.0 - e);
    double K = std::pow(R, 4) + 11 * e * std::pow(R, 5) + 25 * e * e * std::pow(R, 6) + 15 * e * e * e * std::pow(R, 7);
    if (ell) {                                       // 4th derivative of the series: sum k^4 (|C_k| + |S_k|)
        long double C[8], S[8];
        ell_coefficients(e, C, S);
        K = 0.0;
        for (int k = 1; k <= 7; ++k) K += std::pow((double)k, 4) * (double)(fabsl(C[k]) + fabsl(S[k]));
    }
    int l = 7;
    for (; l > 0; --l) {
        const double hw = std::ldexp(w, l);
        if (hw * hw * hw * hw / 384.0 * tau_over_tsamp * K <= 2e-11) break;
    }
    return l;
}

int validate_template(const tb_template& t, double tsamp, std::string* why)
{
    auto bad = [&](const char* m) { *why = m; return TB_ERR_INVALID_ARG; };
    if (!std::isfinite(t.p_orb_s) || t.p_orb_s <= 0) return bad("template: p_orb_s must be finite and > 0");
    if (!std::isfinite(t.tau_lts) || t.tau_lts < 0) return bad("template: tau_lts must be finite and >= 0");
    if (!std::isfinite(t.phi0_rad) || !std::isfinite(t.omega_rad)) return bad("template: phi0/omega must be finite");
    if (!(t.ecc >= 0 && t.ecc < 1)) return bad("template: ecc must be in [0, 1)");
    if (2.0 * t.tau_lts * (1 + t.ecc) / tsamp >= 1073741824.0) return bad("template: shift exceeds 2^30 samples");
    return TB_OK;
}

// knot spacing of one template (the same expressions as make_tmpl, without the trigonometry)
int tmpl_log2h(const tb_template& t, double tsamp, bool ell)
{
    const long double two_pi = 8.0L * atanl(1.0L);
    const long double c = (long double)tsamp / (long double)t.p_orb_s;
    const long double g = (long double)t.tau_lts / (long double)tsamp;
    return knot_log2((double)g, (double)(two_pi * c), t.ecc, ell);
}

// step a1, in long double so that the constants are correctly rounded doubles
void make_tmpl(const tb_template& t, double tsamp, TmplDev* o, EllCoef* ell = nullptr)
{
    const long double two_pi = 8.0L * atanl(1.0L);
    const long double c = (long double)tsamp / (long double)t.p_orb_s;
    o->c_hi = (double)c;
    o->c_lo = (double)(c - (long double)o->c_hi);
    o->w = (double)(two_pi * c);
    long double phi = fmodl((long double)t.phi0_rad, two_pi);
    if (phi < 0) phi += two_pi;
    o->phi0 = (double)phi;
    const long double e = t.ecc, g = (long double)t.tau_lts / (long double)tsamp;
    const long double A = g * sinl((long double)t.omega_rad);
    const long double B = g * sqrtl(1.0L - e * e) * cosl((long double)t.omega_rad);
    o->A = (double)A;
    o->B = (double)B;
    o->ecc = t.ecc;
    o->circular = (t.ecc == 0.0) ? 1 : 0;
    // zero offset: E0 from M = phi0 (Alg. 1)
    const long double M = (long double)o->phi0;
    long double E = M + e * sinl(M);
    for (int it = 0; it < 100; ++it) {
        const long double dE = (E - e * sinl(E) - M) / (1.0L - e * cosl(E));
        E -= dE;
        if (fabsl(dE) < 1e-19L) break;
    }
    o->d0 = (double)((long double)o->A * cosl(E) + (long double)o->B * sinl(E));
    o->log2h = knot_log2((double)g, o->w, t.ecc);
    if (ell) {                                       // ELL7 mode: the S-series carries sqrt(1-e^2); zero offset from the series itself
        long double C[8], S[8];
        ell_coefficients(t.ecc, C, S);
        o->B = (double)(g * cosl((long double)t.omega_rad));
        long double sc = 0.0L, ss = 0.0L;
        for (int k = 1; k <= 7; ++k) {
            ell->c[k - 1] = (double)C[k]; ell->s[k - 1] = (double)S[k];
            sc += (long double)ell->c[k - 1] * cosl((long double)k * M);
            ss += (long double)ell->s[k - 1] * sinl((long double)k * M);
        }
        ell->c[7] = ell->s[7] = 0.0;
        o->d0 = (double)((long double)o->A * sc + (long double)o->B * ss);
        o->circular = 0;
        o->log2h = knot_log2((double)g, o->w, t.ecc, true);
    }
}

// the fill value also sits behind the series, x[N] (4 floats of padding): the fused path clamps an
// out-of-range source index to N instead of testing it again at the gather
int store_fill_pad(tb_plan* p)
{
    for (float& f : p->h_fillpad) f = p->fill;
    TB_CUDA(p, cudaMemcpyAsync(p->d_series_owned + p->n, p->h_fillpad, sizeof(p->h_fillpad), cudaMemcpyHostToDevice, p->stream));
    return TB_OK;
}

struct DevBufs {                                     // scratch of one reduction call, freed on every exit path
    std::vector<void*> ptrs;
    ~DevBufs() { for (void* q : ptrs) cudaFree(q); }
    template <typename T> cudaError_t get(T** out, size_t count)
    {
        void* q = nullptr;
        const cudaError_t e = cudaMalloc(&q, std::max<size_t>(count, 1) * sizeof(T));
        if (e == cudaSuccess) ptrs.push_back(q);
        *out = static_cast<T*>(q);
        return e;
    }
};

int get_fft_plan(tb_plan* p, uint32_t batch, cufftHandle* out);
int run_spectrum(tb_plan* p, uint32_t nt, float* d_raw);

// f2 (reading G25): whiten the plan's copy of the series in place and derive kappa.  Uses the chunk
// scratch (d_fft: spectrum of the series, d_med: block medians), so it runs before any search.
int whiten_series(tb_plan* p)
{
    // double-precision transforms, once per series (see tb_whiten.cuh); the plans are cached
    if (!p->have_c2r) {
        TB_CUFFT(p, cufftPlan1d(&p->d2z_plan, (int)p->n, CUFFT_D2Z, 1));
        cufftResult r = cufftPlan1d(&p->c2r_plan, (int)p->n, CUFFT_Z2D, 1);
        if (r != CUFFT_SUCCESS) { cufftDestroy(p->d2z_plan); return fail(p, r == CUFFT_ALLOC_FAILED ? TB_ERR_NOMEM : TB_ERR_CUFFT, "cufftPlan1d(Z2D)"); }
        p->have_c2r = true;
        TB_CUFFT(p, cufftSetStream(p->d2z_plan, p->stream));
        TB_CUFFT(p, cufftSetStream(p->c2r_plan, p->stream));
    }
    DevBufs mem;
    double* dx = nullptr;
    double2* dX = nullptr;
    TB_CUDA(p, mem.get(&dx, p->n));
    TB_CUDA(p, mem.get(&dX, p->nb + 1));
    k_f32_to_f64<<<1184, 256, 0, p->stream>>>(p->d_series_owned, dx, (size_t)p->n);
    TB_CUFFT(p, cufftExecD2Z(p->d2z_plan, dx, reinterpret_cast<cufftDoubleComplex*>(dX)));
    const unsigned gm = (unsigned)((p->nblk + WH_WARPS - 1) / WH_WARPS);
    switch (p->window) {
        case 128: k_whiten_medians<128><<<gm, WH_WARPS * 32, 0, p->stream>>>(dX, (int)p->nblk, p->d_med); break;
        case 256: k_whiten_medians<256><<<gm, WH_WARPS * 32, 0, p->stream>>>(dX, (int)p->nblk, p->d_med); break;
        case 512: k_whiten_medians<512><<<gm, WH_WARPS * 32, 0, p->stream>>>(dX, (int)p->nblk, p->d_med); break;
        case 1024: k_whiten_medians<1024><<<gm, WH_WARPS * 32, 0, p->stream>>>(dX, (int)p->nblk, p->d_med); break;
        default: k_whiten_medians<2048><<<gm, WH_WARPS * 32, 0, p->stream>>>(dX, (int)p->nblk, p->d_med); break;
    }
    k_whiten_apply<<<(unsigned)((p->nb + 1 + 255) / 256), 256, 0, p->stream>>>(dX, (int)p->nb, (int)p->log2w, (int)p->nblk, p->d_med,
                                                                            1.0 / std::sqrt((double)p->n), p->d_zap, (int)p->zap.size());
    TB_CUDA(p, cudaGetLastError());
    TB_CUFFT(p, cufftExecZ2D(p->c2r_plan, reinterpret_cast<cufftDoubleComplex*>(dX), dx));
    k_f64_to_f32<<<1184, 256, 0, p->stream>>>(dx, p->d_series_owned, (size_t)p->n);
    // kappa from the interbinned spectrum of the whitened, un-resampled series (the production
    // single-precision path: batched R2C + k_spectrum_median): ln2 / mean of its block medians
    cufftHandle r2c;
    if (int rc = get_fft_plan(p, 1, &r2c)) return rc;
    TB_CUFFT(p, cufftExecR2C(r2c, p->d_series_owned, reinterpret_cast<cufftComplex*>(p->d_fft)));
    p->whitening_now = true;
    const int rc = run_spectrum(p, 1, nullptr);
    p->whitening_now = false;
    if (rc) return rc;
    std::vector<float> med(p->nblk);
    TB_CUDA(p, cudaMemcpyAsync(med.data(), p->d_med, p->nblk * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));                // also fences the scratch freed by ~DevBufs
    // blocks touched by a zapped range [lo, hi) (interbinned bins lo..hi) have depressed medians: leave
    // them out of the mean, or kappa grows by 1 / (1 - zapped fraction) (reading G25)
    std::vector<char> keep(p->nblk, 1);
    for (const uint2& z : p->zap)
        for (size_t b = z.x / p->window; b <= z.y / p->window && b < p->nblk; ++b) keep[b] = 0;
    size_t n_keep = 0;
    for (char k : keep) n_keep += k;
    if (n_keep == 0) { std::fill(keep.begin(), keep.end(), 1); n_keep = p->nblk; }
    double acc = 0.0;
    for (size_t b = 0; b < p->nblk; ++b) if (keep[b]) acc += (double)med[b];
    p->kappa = (float)(0.69314718055994530942 * (double)n_keep / acc);
    // the fp64 plans' work areas are several GB from 2^26 samples on and the chunk size B was chosen from
    // the memory free before they existed: give them back (the stream was synchronised above; the next
    // tb_plan_set_series builds them again, milliseconds against the seconds such a series takes to load)
    if (p->n >= (1ull << 26)) {
        cufftDestroy(p->c2r_plan); cufftDestroy(p->d2z_plan);
        p->c2r_plan = p->d2z_plan = 0;
        p->have_c2r = false;
    }
    return TB_OK;
}

// copy the series (from host or device memory) and derive the fill value (G8)
int load_series(tb_plan* p, const float* series)
{
    if (!p->d_series_owned) TB_CUDA(p, cudaMalloc(&p->d_series_owned, (p->n + 4) * sizeof(float)));
    TB_CUDA(p, cudaMemcpyAsync(p->d_series_owned, series, p->n * sizeof(float),
                               p->borrowed ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, p->stream));
    p->d_series = p->d_series_owned;
    if (p->whiten) { const int rc = whiten_series(p); if (rc) return rc; }
    if (p->user_fill) return store_fill_pad(p);
    // fill value (G8): fp64 mean of the series.  296 per-block partial sums on the device (each a
    // fixed strided subset, summed in a fixed order), added up here in block order: deterministic,
    // and the host never walks the series (that loop cost 4 ms of every end-to-end step at 2^23).
    constexpr int SUM_BLOCKS = 296;
    if (!p->d_acc) TB_CUDA(p, cudaMalloc(&p->d_acc, SUM_BLOCKS * sizeof(double)));
    k_sum_f64<<<SUM_BLOCKS, 256, 0, p->stream>>>(p->d_series, (size_t)p->n, p->d_acc);
    TB_CUDA(p, cudaGetLastError());
    double part[SUM_BLOCKS];
    TB_CUDA(p, cudaMemcpyAsync(part, p->d_acc, sizeof(part), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    long double acc = 0.0L;
    for (int i = 0; i < SUM_BLOCKS; ++i) acc += (long double)part[i];
    p->fill = (float)(double)(acc / (long double)p->n);
    return store_fill_pad(p);
}

// Keep the series resident in L2 (persisting access-policy window on the plan's stream): every
// template gathers from the same 4N bytes while tens of GB of scratch stream through the cache.
// Device-wide side effect (documented in tb.h): cudaLimitPersistingL2CacheSize is RAISED to the
// series size if it is smaller, never lowered, and never reset (other plans' windows stay valid).
// On a caller-owned stream the previous window is saved here and restored by destroy().
void pin_series_in_l2(tb_plan* p)
{
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, p->device) != cudaSuccess || prop.persistingL2CacheMaxSize <= 0) return;
    const size_t bytes = std::min<size_t>(p->n * sizeof(float), (size_t)prop.accessPolicyMaxWindowSize);
    const size_t want = std::min<size_t>(bytes, (size_t)prop.persistingL2CacheMaxSize);
    size_t have = 0;
    if (cudaDeviceGetLimit(&have, cudaLimitPersistingL2CacheSize) != cudaSuccess) have = 0;
    if (have < want) cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want);
    // the set-aside actually in force (the call above may have failed or been rounded): a window
    // that asks for more persisting lines than there are only thrashes them
    size_t limit = 0;
    if (cudaDeviceGetLimit(&limit, cudaLimitPersistingL2CacheSize) != cudaSuccess || limit == 0) { cudaGetLastError(); return; }
    if (!p->own_stream && cudaStreamGetAttribute(p->stream, cudaStreamAttributeAccessPolicyWindow, &p->l2_prev) != cudaSuccess)
        std::memset(&p->l2_prev, 0, sizeof(p->l2_prev));
    cudaStreamAttrValue attr;
    std::memset(&attr, 0, sizeof(attr));
    attr.accessPolicyWindow.base_ptr = const_cast<float*>(p->d_series);
    attr.accessPolicyWindow.num_bytes = bytes;
    attr.accessPolicyWindow.hitRatio = std::min(1.0f, (float)limit / (float)bytes);
    attr.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    attr.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    if (cudaStreamSetAttribute(p->stream, cudaStreamAttributeAccessPolicyWindow, &attr) == cudaSuccess) p->l2_pinned = true;
    cudaGetLastError();
}

int get_fft_plan(tb_plan* p, uint32_t batch, cufftHandle* out)
{
    auto it = p->fft_plans.find(batch);
    if (it != p->fft_plans.end()) { *out = it->second; return TB_OK; }
    cufftHandle h;
    TB_CUFFT(p, cufftCreate(&h));
    cufftResult r = cufftSetAutoAllocation(h, 0);
    long long nn[1] = {(long long)p->n};
    long long inembed[1] = {(long long)p->n};
    long long onembed[1] = {(long long)p->ld};
    size_t ws = 0;
    if (r == CUFFT_SUCCESS)
        r = cufftMakePlanMany64(h, 1, nn, inembed, 1, (long long)p->n, onembed, 1, (long long)p->ld, CUFFT_R2C,
                                (long long)batch, &ws);
    if (r != CUFFT_SUCCESS) {
        cufftDestroy(h);
        return fail(p, r == CUFFT_ALLOC_FAILED ? TB_ERR_NOMEM : TB_ERR_CUFFT,
                    "cufftMakePlanMany64 failed: " + std::to_string((int)r));
    }
    if (ws > p->work_bytes) {
        TB_CUDA(p, cudaStreamSynchronize(p->stream));
        if (p->d_work) cudaFree(p->d_work);
        p->d_work = nullptr;
        p->work_bytes = 0;
        cudaError_t e = cudaMalloc(&p->d_work, ws);
        if (e != cudaSuccess) { cufftDestroy(h); return fail(p, TB_ERR_NOMEM, "cuFFT work area allocation failed"); }
        p->work_bytes = ws;
        for (auto& kv : p->fft_plans) TB_CUFFT(p, cufftSetWorkArea(kv.second, p->d_work));
    }
    TB_CUFFT(p, cufftSetWorkArea(h, p->d_work));
    TB_CUFFT(p, cufftSetStream(h, p->stream));
    p->fft_plans[batch] = h;
    *out = h;
    return TB_OK;
}

constexpr int OWN_MIN_LOG2H = 3;                     // the fused path needs >= 2 samples per segment; 8 bounds the table

template <int W>
void launch_spectrum(tb_plan* p, uint32_t nt, float* d_raw)
{
    const int cta_per_row = (int)((p->nblk + SP_WARPS - 1) / SP_WARPS);
    const unsigned grid = (unsigned)(cta_per_row * nt), threads = (SP_WARPS + 1) * 32;
    unsigned long long* fb = p->d_cursor + 1;
    const int nb = (int)p->nb, nblk = (int)p->nblk;
    if (p->over) {                                       // 2x-oversampled spectrum (G12b): nsp = 2 nb half bins
        if (d_raw) k_spectrum_median<W, false, true, false, true><<<grid, threads, 0, p->stream>>>(p->d_fft, p->ld, p->d_power, p->d_med, (int)p->nsp, nblk, cta_per_row, nullptr, nullptr, fb, d_raw, 0.f);
        else       k_spectrum_median<W, false, false, false, true><<<grid, threads, 0, p->stream>>>(p->d_fft, p->ld, p->d_power, p->d_med, (int)p->nsp, nblk, cta_per_row, nullptr, nullptr, fb, nullptr, 0.f);
        return;
    }
    const bool white = p->whiten && !p->whitening_now;   // the whitening procedure itself needs the medians
    if (white) {
        if (d_raw) k_spectrum_median<W, false, true, true><<<grid, threads, 0, p->stream>>>(p->d_fft, p->ld, p->d_power, p->d_med, nb, nblk, cta_per_row, nullptr, nullptr, fb, d_raw, p->kappa);
        else       k_spectrum_median<W, false, false, true><<<grid, threads, 0, p->stream>>>(p->d_fft, p->ld, p->d_power, p->d_med, nb, nblk, cta_per_row, nullptr, nullptr, fb, nullptr, p->kappa);
        return;
    }
    if (d_raw) k_spectrum_median<W, false, true><<<grid, threads, 0, p->stream>>>(p->d_fft, p->ld, p->d_power, p->d_med, nb, nblk, cta_per_row, nullptr, nullptr, fb, d_raw, 0.f);
    else       k_spectrum_median<W, false, false><<<grid, threads, 0, p->stream>>>(p->d_fft, p->ld, p->d_power, p->d_med, nb, nblk, cta_per_row, nullptr, nullptr, fb, nullptr, 0.f);
}

// ---- hand-written FFT path -------------------------------------------------------------------
// columns per CTA of pass 1: 16 (runs of 32 samples / 128 bytes); M1 = 1024 has its own kernel (k_fft_cols1k, 8 columns)
template <int R1, int C> constexpr size_t cols_smem() { return (size_t)(C * (R1 * FFT_PA + 16 / C) + 256) * sizeof(float2); }

template <int R1, int FFT_C, bool DEBUG>
int launch_cols(tb_plan* p, size_t off, uint32_t nt, long long* d_idx, float* d_y)
{
    auto kern = k_fft_cols<R1, FFT_C, DEBUG>;
    if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(kern), (size_t)(cols_smem<R1, FFT_C>()))) return rc_;
    const unsigned grid = (unsigned)(((1u << p->log2m2) / FFT_C) * nt);
    kern<<<grid, FFT_THREADS, cols_smem<R1, FFT_C>(), p->stream>>>(p->d_series, p->d_seg, p->seg_stride, p->d_tmpl + off, (int)nt,
                                                           (int)p->n, p->log2m2, p->fill, p->d_tw1a, p->d_tw2,
                                                           reinterpret_cast<float2*>(p->d_resampled), d_idx, d_y, p->pf_cols);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

template <int R1, bool TWIN = false>
int launch_rows(tb_plan* p, uint32_t nt)
{
    using Cfg = RowsCfg<R1>;
    auto kern = k_fft_rows_t<R1, TWIN>;
    if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(kern), (size_t)(Cfg::SMEM))) return rc_;
    const unsigned grid = (unsigned)(((1u << p->log2m1) / Cfg::R) * nt);
    kern<<<grid, FFT_THREADS, Cfg::SMEM, p->stream>>>(reinterpret_cast<const float2*>(p->d_resampled), p->d_fft, p->log2m1,
                                                     p->d_tw1b, p->d_tw2, p->pf_rows);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

// N = 2^23 (rows of 8192 points): the four-step twiddle is applied by pass 2 on load instead of pass 1 on store
bool twiddle_in_pass2(const tb_plan* p) { return p->cols32 && p->log2m2 == 13; }

template <bool DEBUG>
int launch_cols32(tb_plan* p, size_t off, uint32_t nt, long long* d_idx, float* d_y)
{
    auto kern = twiddle_in_pass2(p) ? k_fft_cols32<DEBUG, false> : k_fft_cols32<DEBUG, true>;
    if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(kern), (size_t)(C32_SMEM))) return rc_;
    const unsigned grid = (unsigned)(((1u << p->log2m2) / 16) * nt);
    kern<<<grid, FFT_THREADS, C32_SMEM, p->stream>>>(p->d_series, p->d_seg, p->seg_stride, p->d_tmpl + off, (int)nt, (int)p->n,
                                                    p->log2m2, p->fill, p->d_twc, reinterpret_cast<float2*>(p->d_resampled),
                                                    d_idx, d_y, p->pf_cols);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

template <bool DEBUG>
int launch_cols1k(tb_plan* p, size_t off, uint32_t nt, long long* d_idx, float* d_y)
{
    auto kern = k_fft_cols1k<DEBUG>;
    if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(kern), (size_t)(C1K_SMEM))) return rc_;
    const unsigned grid = (unsigned)(((1u << p->log2m2) / 8) * nt);
    kern<<<grid, FFT_THREADS, C1K_SMEM, p->stream>>>(p->d_series, p->d_seg, p->seg_stride, p->d_tmpl + off, (int)nt, (int)p->n,
                                                    p->log2m2, p->fill, p->d_twc, reinterpret_cast<float2*>(p->d_resampled),
                                                    d_idx, d_y, p->pf_cols);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

// K0 + P1: delay segments, then gather + column FFTs into T (the buffer the legacy path uses for y)
int run_k0(tb_plan* p, size_t off, uint32_t nt, cudaStream_t st)
{
    const int cta_per_tmpl = (int)(((p->n >> p->chunk_log2h) + 255) / 256);   // chunk_log2h: smallest knot spacing in this chunk
    k_delay_segments<<<(unsigned)(cta_per_tmpl * nt), K0_THREADS, 0, st>>>(p->d_tmpl + off, (int)nt, (int)p->n, p->d_seg,
                                                                    p->seg_stride, cta_per_tmpl, p->ell ? p->d_ell + off : nullptr);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

int run_p1(tb_plan* p, size_t off, uint32_t nt, long long* d_idx, float* d_y);

int run_own_pass1(tb_plan* p, size_t off, uint32_t nt, long long* d_idx, float* d_y)
{
    if (int rc = run_k0(p, off, nt, p->stream)) return rc;
    return run_p1(p, off, nt, d_idx, d_y);
}

int run_p1(tb_plan* p, size_t off, uint32_t nt, long long* d_idx, float* d_y)
{
    const bool dbg = d_idx != nullptr;
    if (p->cols32) return dbg ? launch_cols32<true>(p, off, nt, d_idx, d_y) : launch_cols32<false>(p, off, nt, nullptr, nullptr);
    switch (p->log2m1 - 8) {
        case 0: return dbg ? launch_cols<1, 16, true>(p, off, nt, d_idx, d_y) : launch_cols<1, 16, false>(p, off, nt, nullptr, nullptr);
        case 2: return dbg ? launch_cols1k<true>(p, off, nt, d_idx, d_y) : launch_cols1k<false>(p, off, nt, nullptr, nullptr);
    }
    return fail(p, TB_ERR_INVALID_ARG, "unsupported M1");
}

// three-pass FFT (N >= 2^25): rows of M2 = 2^16 = 256 x 256 points, in place over the slow index, then scattered rows
int run_own_pass23(tb_plan* p, uint32_t nt)
{
    const unsigned rows = nt << p->log2m1;
    {
        auto kern = k_fft_cols<1, 16, false, true>;
        if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(kern), (size_t)(cols_smem<1, 16>()))) return rc_;
        kern<<<rows * 16, FFT_THREADS, cols_smem<1, 16>(), p->stream>>>(nullptr, nullptr, 0, nullptr, (int)rows, 0, 8, 0.f, p->d_tw1b, p->d_tw2,
                                                                       reinterpret_cast<float2*>(p->d_resampled), nullptr, nullptr, p->pf_mid);
        TB_CUDA(p, cudaGetLastError());
    }
    {
        if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(k_fft_rows_scatter), (size_t)(RS_SMEM))) return rc_;
        k_fft_rows_scatter<<<rows * 16, FFT_THREADS, RS_SMEM, p->stream>>>(reinterpret_cast<const float2*>(p->d_resampled), p->d_fft, p->d_tw2, p->pf_scat);
        TB_CUDA(p, cudaGetLastError());
    }
    return TB_OK;
}

// rows of 16384 points (N = 2^24): one CTA of 512 threads per row
int launch_rows_wide(tb_plan* p, uint32_t nt)
{
    if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(k_fft_rows_wide), RW_SMEM)) return rc_;
    const unsigned grid = (unsigned)(nt << p->log2m1);
    k_fft_rows_wide<<<grid, RW_THREADS, RW_SMEM, p->stream>>>(reinterpret_cast<const float2*>(p->d_resampled), p->d_fft, p->d_tw1b,
                                                              p->d_tw512, p->n_sm);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

int run_own_pass2(tb_plan* p, uint32_t nt)
{
    if (p->log2m2 == 16) return run_own_pass23(p, nt);
    if (p->log2m2 == 14) return launch_rows_wide(p, nt);
    switch (p->log2m2 - 8) {
        case 0: return launch_rows<1>(p, nt);
        case 1: return launch_rows<2>(p, nt);
        case 2: return launch_rows<4>(p, nt);
        case 3: return launch_rows<8>(p, nt);
        case 4: return launch_rows<16>(p, nt);
        case 5: return twiddle_in_pass2(p) ? launch_rows<32, true>(p, nt) : launch_rows<32>(p, nt);
    }
    return fail(p, TB_ERR_INVALID_ARG, "unsupported M2");
}

template <int W, int LOG2M1, bool RAW, bool WHITE>
int launch_spectrum_t1(tb_plan* p, uint32_t nt, float* d_raw)
{
    constexpr size_t smem = st_smem_bytes(W, LOG2M1);
    const unsigned grid = (unsigned)((p->nblk / 16) * nt);
    auto kern = k_spectrum_t<W, LOG2M1, RAW, WHITE>;
    if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(kern), (size_t)(smem))) return rc_;
    kern<<<grid, ST_THREADS, smem, p->stream>>>(p->d_fft, p->d_power, p->d_med, p->log2m2, (int)p->nblk, p->d_twn, p->d_twb, p->rot,
                                                p->d_cursor + 1, d_raw, p->pf_spec, p->kappa);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

template <int W, int LOG2M1>
int launch_spectrum_t(tb_plan* p, uint32_t nt, float* d_raw)
{
    if (p->whiten) return d_raw ? launch_spectrum_t1<W, LOG2M1, true, true>(p, nt, d_raw) : launch_spectrum_t1<W, LOG2M1, false, true>(p, nt, nullptr);
    return d_raw ? launch_spectrum_t1<W, LOG2M1, true, false>(p, nt, d_raw) : launch_spectrum_t1<W, LOG2M1, false, false>(p, nt, nullptr);
}

// (median window, log2 M1) pairs the transposing spectrum former is instantiated for
bool spectrum_t_supported(uint32_t w, int log2m1)
{
    return (log2m1 == 8 && (w == 256 || w == 1024)) || (log2m1 == 9 && (w == 512 || w == 1024 || w == 2048)) ||
           (log2m1 == 10 && (w == 1024 || w == 2048));
}

int run_spectrum_t(tb_plan* p, uint32_t nt, float* d_raw = nullptr)
{
    switch (p->window * 16 + (uint32_t)p->log2m1) {
        case 256 * 16 + 8: return launch_spectrum_t<256, 8>(p, nt, d_raw);
        case 1024 * 16 + 8: return launch_spectrum_t<1024, 8>(p, nt, d_raw);
        case 512 * 16 + 9: return launch_spectrum_t<512, 9>(p, nt, d_raw);
        case 1024 * 16 + 9: return launch_spectrum_t<1024, 9>(p, nt, d_raw);
        case 2048 * 16 + 9: return launch_spectrum_t<2048, 9>(p, nt, d_raw);
        case 1024 * 16 + 10: return launch_spectrum_t<1024, 10>(p, nt, d_raw);
        case 2048 * 16 + 10: return launch_spectrum_t<2048, 10>(p, nt, d_raw);
    }
    return fail(p, TB_ERR_INVALID_ARG, "median_window");
}

// twiddle tables of the hand-written FFT, in long double, rounded once to fp32
int make_twiddles(tb_plan* p)
{
    const long double two_pi = 8.0L * atanl(1.0L);
    auto upload = [&](std::vector<float2>& h, float2** d) -> int {
        TB_CUDA(p, cudaMalloc(d, h.size() * sizeof(float2)));
        TB_CUDA(p, cudaMemcpy(*d, h.data(), h.size() * sizeof(float2), cudaMemcpyHostToDevice));
        return TB_OK;
    };
    auto tw1 = [&](int log2l, float2** d) -> int {       // [ka*256 + w] = W_L^{w ka}
        const int L = 1 << log2l, R1 = L / 256;
        std::vector<float2> h((size_t)L);
        for (int ka = 0; ka < R1; ++ka)
            for (int w = 0; w < 256; ++w) {
                const long double a = -two_pi * (long double)((long long)w * ka % L) / (long double)L;
                h[(size_t)ka * 256 + w] = make_float2((float)cosl(a), (float)sinl(a));
            }
        return upload(h, d);
    };
    int rc;
    if ((rc = tw1(p->log2m1, &p->d_tw1a))) return rc;
    if (p->log2m2 == 14) {                               // k_fft_rows_wide: W_L^w, W_L^{8w} (L = 16384, w < 512) and W_512^{c kb}
        std::vector<float2> h(1024), h5(512);
        for (int w = 0; w < 512; ++w) {
            const long double a1 = -two_pi * (long double)w / 16384.0L, a8 = -two_pi * (long double)(8 * w) / 16384.0L;
            h[w] = make_float2((float)cosl(a1), (float)sinl(a1));
            h[512 + w] = make_float2((float)cosl(a8), (float)sinl(a8));
        }
        for (int kb = 0; kb < 16; ++kb)
            for (int c = 0; c < 32; ++c) {
                const long double a = -two_pi * (long double)(kb * c) / 512.0L;
                h5[kb * 32 + c] = make_float2((float)cosl(a), (float)sinl(a));
            }
        if ((rc = upload(h, &p->d_tw1b))) return rc;
        if ((rc = upload(h5, &p->d_tw512))) return rc;
    } else if ((rc = tw1(p->log2m2 == 16 ? 8 : p->log2m2, &p->d_tw1b))) return rc;
    std::vector<float2> h2(256), hn((size_t)1 << p->log2m1), hb((size_t)1 << p->log2m2);
    for (int kb = 0; kb < 16; ++kb)
        for (int c = 0; c < 16; ++c) {
            const long double a = -two_pi * (long double)(kb * c) / 256.0L;
            h2[kb * 16 + c] = make_float2((float)cosl(a), (float)sinl(a));
        }
    for (size_t i = 0; i < hn.size(); ++i) {             // R2C twiddle W_N^k = W_N^{k1} * W_N^{M1 k2}
        const long double a = -two_pi * (long double)i / (long double)p->n;
        hn[i] = make_float2((float)cosl(a), (float)sinl(a));
    }
    for (size_t b = 0; b < hb.size(); ++b) {
        const long double a = -two_pi * (long double)((uint64_t)b << p->log2m1) / (long double)p->n;
        hb[b] = make_float2((float)cosl(a), (float)sinl(a));
    }
    if (p->log2m1 == 10) {                               // W_1024^{c ka} of the 32 x 32 first pass
        std::vector<float2> hc(1024);
        for (int ka = 0; ka < 32; ++ka)
            for (int c = 0; c < 32; ++c) {
                const long double a = -two_pi * (long double)(ka * c) / 1024.0L;
                hc[ka * 32 + c] = make_float2((float)cosl(a), (float)sinl(a));
            }
        if ((rc = upload(hc, &p->d_twc))) return rc;
    }
    if (p->log2m1 == 9) {                                // W_512^{c ka} of the 32 x 16 first pass
        std::vector<float2> hc(512);
        for (int ka = 0; ka < 32; ++ka)
            for (int c = 0; c < 16; ++c) {
                const long double a = -two_pi * (long double)(ka * c) / 512.0L;
                hc[ka * 16 + c] = make_float2((float)cosl(a), (float)sinl(a));
            }
        if ((rc = upload(hc, &p->d_twc))) return rc;
        p->cols32 = true;
    }
    p->rot = make_float2((float)cosl(two_pi / (long double)p->n), (float)-sinl(two_pi / (long double)p->n));
    if ((rc = upload(h2, &p->d_tw2))) return rc;
    if ((rc = upload(hb, &p->d_twb))) return rc;
    return upload(hn, &p->d_twn);
}

// stages of one chunk of nt templates whose constants sit at d_tmpl + off
int run_resample(tb_plan* p, size_t off, uint32_t nt, long long* d_idx)
{
    const int tile = (int)std::min<uint64_t>(RS_TILE, p->n);
    const unsigned grid = (unsigned)((p->n / tile) * nt);
    if (d_idx)
        k_resample<true><<<grid, RS_THREADS, 0, p->stream>>>(p->d_series, p->d_resampled, p->d_tmpl + off, (int)nt,
                                                             (int)p->n, tile, p->fill, d_idx, p->ell ? p->d_ell + off : nullptr);
    else
        k_resample<false><<<grid, RS_THREADS, 0, p->stream>>>(p->d_series, p->d_resampled, p->d_tmpl + off, (int)nt,
                                                              (int)p->n, tile, p->fill, nullptr, p->ell ? p->d_ell + off : nullptr);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

int run_fft(tb_plan* p, uint32_t nt)
{
    cufftHandle h;
    int rc = get_fft_plan(p, nt, &h);
    if (rc) return rc;
    TB_CUFFT(p, cufftExecR2C(h, p->d_resampled, reinterpret_cast<cufftComplex*>(p->d_fft)));
    return TB_OK;
}

int run_spectrum(tb_plan* p, uint32_t nt, float* d_raw)
{
    switch (p->window) {
        case 128: launch_spectrum<128>(p, nt, d_raw); break;
        case 256: launch_spectrum<256>(p, nt, d_raw); break;
        case 512: launch_spectrum<512>(p, nt, d_raw); break;
        case 1024: launch_spectrum<1024>(p, nt, d_raw); break;
        case 2048: launch_spectrum<2048>(p, nt, d_raw); break;
        default: return fail(p, TB_ERR_INVALID_ARG, "median_window");
    }
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

// a8 + a9 for the nt templates at d_tmpl + off (their ids come from TmplDev::id); tap: parity tap [5][nb] or null
int run_hsum(tb_plan* p, size_t off, uint32_t nt, const FoldParams& fp, float* tap = nullptr)
{
    const TmplDev* tm = p->d_tmpl + off;
    if (p->nsp >= (uint64_t)HS_T) {
        const int tiles = (int)(p->nsp / HS_T);
        const int tpc = std::min(tiles, HS_TPC);                                     // tiles walked by one CTA (double-buffered)
        const size_t smem = HS_BUFS * HS_SMEM_FLOATS * sizeof(float);
        const unsigned grid = (unsigned)((tiles / tpc) * nt);
        if (tap) {
            if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(k_hsum_tile<true>), smem)) return rc_;
            k_hsum_tile<true><<<grid, HS_THREADS, smem, p->stream>>>(p->d_power, (int)p->nsp, tiles / tpc, tpc, fp, tm, p->d_cand, p->d_cursor,
                                                                    (unsigned long long)p->max_cand, tap);
        } else {
            if (int rc_ = allow_smem(p, reinterpret_cast<const void*>(k_hsum_tile<false>), smem)) return rc_;
            k_hsum_tile<false><<<grid, HS_THREADS, smem, p->stream>>>(p->d_power, (int)p->nsp, tiles / tpc, tpc, fp, tm, p->d_cand, p->d_cursor,
                                                                     (unsigned long long)p->max_cand, nullptr);
        }
        TB_CUDA(p, cudaGetLastError());
        return TB_OK;
    }
    const int cta_per_row = (int)((p->nsp + 255) / 256);
    if (tap) k_hsum_threshold<true><<<(unsigned)(cta_per_row * nt), 256, 0, p->stream>>>(p->d_power, (int)p->nsp, cta_per_row, fp, tm, p->d_cand,
                                                                                     p->d_cursor, (unsigned long long)p->max_cand, tap);
    else     k_hsum_threshold<false><<<(unsigned)(cta_per_row * nt), 256, 0, p->stream>>>(p->d_power, (int)p->nsp, cta_per_row, fp, tm, p->d_cand,
                                                                                      p->d_cursor, (unsigned long long)p->max_cand, nullptr);
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

// the fused path needs records of >= 8 samples; the rest of a bank goes through k_resample + cuFFT

// Validate the bank, size the staging buffers, and split it by launch sequence (stable partition:
// templates the fused path can take first, the others after them), so that one fast-orbit template
// does not send the whole bank through the library-FFT path.  p->order[pos] = index in the caller's
// array of the template staged at position pos; the candidates carry first_id + that index.
int upload_templates(tb_plan* p, const tb_template* tmpl, uint64_t k)
{
    for (uint64_t i = 0; i < k; ++i) {
        std::string why;
        if (validate_template(tmpl[i], p->tsamp, &why)) return fail(p, TB_ERR_INVALID_ARG, why + " (index " + std::to_string(i) + ")");
    }
    if (p->staged_pending) {
        TB_CUDA(p, cudaEventSynchronize(p->ev_staged));
        p->staged_pending = false;
    }
    if (k > p->h_tmpl_cap) {
        if (p->h_tmpl) cudaFreeHost(p->h_tmpl);
        p->h_tmpl = nullptr; p->h_tmpl_cap = 0;
        TB_CUDA(p, cudaMallocHost(&p->h_tmpl, k * sizeof(TmplDev)));
        if (p->ell) {
            if (p->h_ell) cudaFreeHost(p->h_ell);
            p->h_ell = nullptr;
            TB_CUDA(p, cudaMallocHost(&p->h_ell, k * sizeof(EllCoef)));
        }
        p->h_tmpl_cap = k;
    }
    if (k > p->tmpl_cap) {
        TB_CUDA(p, cudaStreamSynchronize(p->stream));
        if (p->d_tmpl) cudaFree(p->d_tmpl);
        p->d_tmpl = nullptr; p->tmpl_cap = 0;
        TB_CUDA(p, cudaMalloc(&p->d_tmpl, k * sizeof(TmplDev)));
        if (p->ell) {
            if (p->d_ell) cudaFree(p->d_ell);
            p->d_ell = nullptr;
            TB_CUDA(p, cudaMalloc(&p->d_ell, k * sizeof(EllCoef)));
        }
        p->tmpl_cap = k;
    }
    // knot spacings first (cheap): they select the launch sequence of every template and the size of
    // the segment table; the constants themselves are made and uploaded chunk by chunk (stage_chunk),
    // so that the host's extended-precision trigonometry overlaps the kernels of the previous chunk
    p->order.resize(k);
    std::vector<uint32_t> rest;
    size_t n_own = 0;
    int min_own = 7;
    for (uint64_t i = 0; i < k; ++i) {
        const int l = p->own_fft ? tmpl_log2h(tmpl[i], p->tsamp, p->ell) : 0;
        if (p->own_fft && l >= OWN_MIN_LOG2H) { p->order[n_own++] = (uint32_t)i; min_own = std::min(min_own, l); }
        else rest.push_back((uint32_t)i);
    }
    std::copy(rest.begin(), rest.end(), p->order.begin() + n_own);
    p->n_own = n_own;
    if (n_own) {                                         // segment table: chunk x (n >> smallest spacing) records
        p->seg_stride = (size_t)(p->n >> min_own);
        const size_t need = (size_t)std::min<uint64_t>(p->chunk, n_own) * p->seg_stride;
        if (need > p->seg_cap) {
            TB_CUDA(p, cudaStreamSynchronize(p->stream));
            if (p->d_seg) cudaFree(p->d_seg);
            p->d_seg = nullptr; p->seg_cap = 0;
            TB_CUDA(p, cudaMalloc(&p->d_seg, need * sizeof(SegRec)));
            p->seg_cap = need;
        }
    }
    return TB_OK;
}

// constants of the templates staged at positions [off, off + nt), uploaded on the plan's stream
int stage_chunk(tb_plan* p, const tb_template* tmpl, uint64_t off, uint64_t nt, uint32_t first_id, cudaStream_t st)
{
    int lmin = 7;
    for (uint64_t i = off; i < off + nt; ++i) {
        make_tmpl(tmpl[p->order[i]], p->tsamp, &p->h_tmpl[i], p->ell ? &p->h_ell[i] : nullptr);
        p->h_tmpl[i].id = first_id + p->order[i];
        p->h_tmpl[i].pad = 0;
        lmin = std::min(lmin, p->h_tmpl[i].log2h);
    }
    p->chunk_log2h = lmin;
    TB_CUDA(p, cudaMemcpyAsync(p->d_tmpl + off, p->h_tmpl + off, nt * sizeof(TmplDev), cudaMemcpyHostToDevice, st));
    if (p->ell) TB_CUDA(p, cudaMemcpyAsync(p->d_ell + off, p->h_ell + off, nt * sizeof(EllCoef), cudaMemcpyHostToDevice, st));
    // recorded after EVERY chunk: whatever way the call ends, the next one waits for the last copy
    // out of the pinned staging buffer before it rewrites it
    TB_CUDA(p, cudaEventRecord(p->ev_staged, st));
    p->staged_pending = true;
    return TB_OK;
}

int make_fold_params(tb_plan* p, const uint32_t* folds, uint32_t n_folds, double sigma, FoldParams* fp)
{
    if (!std::isfinite(sigma)) return fail(p, TB_ERR_INVALID_ARG, "sigma_threshold must be finite");
    if (n_folds > 0 && !folds) return fail(p, TB_ERR_INVALID_ARG, "folds is NULL");
    bool seen[5] = {false, false, false, false, false};
    for (uint32_t i = 0; i < n_folds; ++i) {
        if (folds[i] > TB_MAX_FOLD) return fail(p, TB_ERR_INVALID_ARG, "fold > 4");
        if (seen[folds[i]]) return fail(p, TB_ERR_INVALID_ARG, "duplicate fold");
        seen[folds[i]] = true;
    }
    for (uint32_t L = 0; L < 5; ++L) {
        double mu, s;
        sigma_constants(L, &mu, &s);
        fp->mu[L] = (float)mu;
        fp->inv_s[L] = (float)(1.0 / s);
        const double root = mu + sigma * s;
        fp->thr[L] = seen[L] ? (root <= 0 ? 0.f : (float)(root * root)) : std::numeric_limits<float>::infinity();
    }
    for (uint32_t L = 0; L < 5; ++L) fp->lo[L] = (uint32_t)std::min<uint64_t>((uint64_t)p->k_lo << L, p->nsp);
    return TB_OK;
}

void destroy(tb_plan* p)
{
    if (!p) return;
    cudaSetDevice(p->device);
    if (p->stream) cudaStreamSynchronize(p->stream);
    if (p->l2_pinned && !p->own_stream)              // give a caller-owned stream its previous window back
        cudaStreamSetAttribute(p->stream, cudaStreamAttributeAccessPolicyWindow, &p->l2_prev);
    for (auto& kv : p->fft_plans) cufftDestroy(kv.second);
    if (p->have_c2r) { cufftDestroy(p->c2r_plan); cufftDestroy(p->d2z_plan); }
    cudaFree(p->d_zap);
    for (auto& es : p->events) for (auto& e : es.e) cudaEventDestroy(e);
    if (p->s_k0) { cudaStreamSynchronize(p->s_k0); cudaStreamDestroy(p->s_k0); }
    for (auto& es : p->events) for (auto& e : es.k) cudaEventDestroy(e);
    if (p->ev_staged) cudaEventDestroy(p->ev_staged);
    if (p->ev_main) cudaEventDestroy(p->ev_main);
    if (p->ev_p1) cudaEventDestroy(p->ev_p1);
    if (p->ev_k0) cudaEventDestroy(p->ev_k0);
    cudaFree(p->d_seg); cudaFree(p->d_tw512); cudaFree(p->d_tw1a); cudaFree(p->d_tw1b); cudaFree(p->d_tw2); cudaFree(p->d_twn); cudaFree(p->d_twb); cudaFree(p->d_twc);
    cudaFree(p->d_work); cudaFree(p->d_acc); cudaFree(p->d_series_owned); cudaFree(p->d_resampled); cudaFree(p->d_fft);
    cudaFree(p->d_power); cudaFree(p->d_med); cudaFree(p->d_cand); cudaFree(p->d_cursor); cudaFree(p->d_tmpl);
    if (p->h_tmpl) cudaFreeHost(p->h_tmpl);
    if (p->h_ell) cudaFreeHost(p->h_ell);
    cudaFree(p->d_ell);
    if (p->own_stream && p->stream) cudaStreamDestroy(p->stream);
    delete p;
}

int single_template_stage(tb_plan* p, const tb_template* tmpl)
{
    if (!p || !tmpl) return fail(p, TB_ERR_INVALID_ARG, "null argument");
    TB_CUDA(p, cudaSetDevice(p->device));
    const int rc = upload_templates(p, tmpl, 1);
    return rc ? rc : stage_chunk(p, tmpl, 0, 1, 0, p->stream);
}

}  // namespace

extern "C" {

const char* tb_strerror(int code)
{
    switch (code) {
        case TB_OK: return "ok";
        case TB_ERR_INVALID_ARG: return "invalid argument";
        case TB_ERR_CUDA: return "CUDA error";
        case TB_ERR_CUFFT: return "cuFFT error";
        case TB_ERR_NOMEM: return "out of memory";
        case TB_ERR_OVERFLOW: return "candidate buffer overflow";
        case TB_ERR_CAPACITY: return "output buffer too small";
        default: return "unknown error";
    }
}

const char* tb_last_error(const tb_plan* plan) { return plan ? plan->err.c_str() : "null plan"; }

int tb_sigma_to_power(uint32_t fold, double sigma, double* power_out)
{
    if (fold > TB_MAX_FOLD || !power_out || !std::isfinite(sigma)) return TB_ERR_INVALID_ARG;
    double mu, s;
    sigma_constants(fold, &mu, &s);
    const double r = mu + sigma * s;
    *power_out = r <= 0 ? 0.0 : r * r;
    return TB_OK;
}

int tb_plan_create(tb_plan** out, const float* series, uint64_t n_samples, double tsamp_s, const tb_plan_opts* uopts)
{
    if (!out) return TB_ERR_INVALID_ARG;
    *out = nullptr;
    tb_plan_opts o;
    std::memset(&o, 0, sizeof(o));
    if (uopts) {
        if (uopts->struct_size < 8 || uopts->struct_size > sizeof(o)) return TB_ERR_INVALID_ARG;
        std::memcpy(&o, uopts, uopts->struct_size);
    }
    const uint32_t W = o.median_window ? o.median_window : 1024;
    if (!series || !(tsamp_s > 0) || !std::isfinite(tsamp_s)) return TB_ERR_INVALID_ARG;
    if (!is_pow2(W) || W < 128 || W > 2048) return TB_ERR_INVALID_ARG;
    if (!is_pow2(n_samples) || n_samples < 2ull * W || n_samples > (1ull << 28)) return TB_ERR_INVALID_ARG;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || o.device < 0 || o.device >= ndev) return TB_ERR_CUDA;

    tb_plan* p = new (std::nothrow) tb_plan;
    if (!p) return TB_ERR_NOMEM;
    p->device = o.device;
    p->n = n_samples;
    p->nb = n_samples / 2;
    p->tsamp = tsamp_s;
    p->window = W;
    p->log2w = ilog2(W);
    p->over = o.interbin_oversample != 0;
    if (o.interbin_oversample != 0 && o.interbin_oversample != 1) { delete p; return TB_ERR_INVALID_ARG; }
    if (p->over && (o.whiten || n_samples > (1ull << 27))) { delete p; return TB_ERR_INVALID_ARG; }   // no whitened variant; 2 nb must fit the 32-bit bin index
    p->nsp = p->over ? 2 * p->nb : p->nb;
    p->nblk = (uint32_t)(p->nsp / W);
    p->f_min = (o.f_min_hz == 0.0) ? 0.1 : (o.f_min_hz < 0 ? 0.0 : o.f_min_hz);
    p->k_lo = (uint32_t)std::min<double>(std::ceil(p->f_min * ((double)n_samples * tsamp_s)) * (p->over ? 2.0 : 1.0), 4294967295.0);   // half bins when oversampled
    p->max_cand = o.max_candidates ? o.max_candidates : (1ull << 22);
    p->timings = o.enable_timings != 0;
    p->whiten = o.whiten != 0;
    if (o.delay_model != 0 && o.delay_model != 1) { delete p; return TB_ERR_INVALID_ARG; }
    p->ell = o.delay_model == 1;
    if (o.n_zap_ranges) {
        if (!o.zap_ranges) { delete p; return TB_ERR_INVALID_ARG; }
        for (uint32_t z = 0; z < o.n_zap_ranges; ++z) {
            const uint32_t lo = o.zap_ranges[2 * z], hi = o.zap_ranges[2 * z + 1];
            if (lo >= hi || hi > n_samples / 2) { delete p; return TB_ERR_INVALID_ARG; }
            p->zap.push_back(make_uint2(lo, hi));
        }
    }
    p->ld = p->nb + 4;                                // N/2+1 bins padded to a multiple of 4 complex (32 B)

    auto bail = [&](int code, const std::string& m) { (void)m; destroy(p); return code; };
#define TB_TRY(call)                                                                                   \
    do {                                                                                               \
        cudaError_t e__ = (call);                                                                      \
        if (e__ != cudaSuccess)                                                                        \
            return bail(e__ == cudaErrorMemoryAllocation ? TB_ERR_NOMEM : TB_ERR_CUDA, #call);         \
    } while (0)

    TB_TRY(cudaSetDevice(p->device));
    if (o.stream) p->stream = (cudaStream_t)o.stream;
    else { TB_TRY(cudaStreamCreateWithFlags(&p->stream, cudaStreamNonBlocking)); p->own_stream = true; }
    TB_TRY(cudaEventCreateWithFlags(&p->ev_staged, cudaEventDisableTiming));
    TB_TRY(cudaStreamCreateWithFlags(&p->s_k0, cudaStreamNonBlocking));
    TB_TRY(cudaEventCreateWithFlags(&p->ev_main, cudaEventDisableTiming));
    TB_TRY(cudaEventCreateWithFlags(&p->ev_p1, cudaEventDisableTiming));
    TB_TRY(cudaEventCreateWithFlags(&p->ev_k0, cudaEventDisableTiming));

    // chunk size B
    const size_t per_t = (size_t)p->n * 4 + p->ld * 8 + (size_t)p->nsp * 4 + (size_t)p->nblk * 4 + (size_t)p->n * 8;
    uint32_t B = o.chunk_templates;
    if (B == 0) {
        size_t free_b = 0, total_b = 0;
        TB_TRY(cudaMemGetInfo(&free_b, &total_b));
        const uint64_t by_size = std::max<uint64_t>(1, (1ull << 29) / p->n);
        const uint64_t by_mem = std::max<uint64_t>(1, (uint64_t)(0.5 * (double)free_b) / (per_t * 2));   // x2: cuFFT work area
        B = (uint32_t)std::min<uint64_t>(std::min<uint64_t>(by_size, by_mem), 256);
    }
    p->chunk = B;

    p->borrowed = o.series_is_device_ptr != 0;
    p->user_fill = o.has_fill != 0;
    p->fill = o.fill_value;

    // FFT path: hand-written two-pass FFT (M = N/2 = M1 * M2, M1 = 512, 256 at 2^17, 1024 at 2^25) when
    // 2^17 <= N <= 2^26 (three passes with M2 = 256 x 256 at 2^26), W >= M1 and the median blocks pair up in groups of 16; batched cuFFT otherwise
    {
        const int lm = (int)ilog2(p->nb);
        p->log2m1 = lm == 24 ? 10 : lm >= 17 ? 9 : 8;   // 2^24, 2^25: rows of 16384 (k_fft_rows_wide) with M1 = 512, 1024; 2^26: three passes, M2 = 2^16
        p->log2m2 = lm - p->log2m1;
        const bool fits = ((p->log2m2 >= 8 && p->log2m2 <= 14) || (p->log2m2 == 16 && lm >= 24)) && spectrum_t_supported(W, p->log2m1) && p->nblk >= 16 && p->nblk % 16 == 0;
        if (o.fft_path >= 2 && (!fits || p->over)) { destroy(p); return TB_ERR_INVALID_ARG; }
        p->own_fft = fits && o.fft_path != 1 && !p->over;         // the oversampled spectrum is formed from the library R2C output
    }
    if (p->own_fft) {
        cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, p->device);
        p->pf_rows = p->n_sm * 2;
        int rc = make_twiddles(p);
        if (rc) { destroy(p); return rc; }
    }
    TB_TRY(cudaMalloc(&p->d_resampled, (size_t)B * p->n * sizeof(float)));
    TB_TRY(cudaMalloc(&p->d_fft, (size_t)B * p->ld * sizeof(float2)));
    TB_TRY(cudaMalloc(&p->d_power, (size_t)B * p->nsp * sizeof(float)));
    TB_TRY(cudaMalloc(&p->d_med, (size_t)B * p->nblk * sizeof(float)));
    TB_TRY(cudaMalloc(&p->d_cand, p->max_cand * sizeof(Candidate)));
    TB_TRY(cudaMalloc(&p->d_cursor, 2 * sizeof(unsigned long long)));   // [0] candidate cursor, [1] median fallbacks
    TB_TRY(cudaMemsetAsync(p->d_cursor, 0, 2 * sizeof(unsigned long long), p->stream));
    if (!p->zap.empty()) {
        TB_TRY(cudaMalloc(&p->d_zap, p->zap.size() * sizeof(uint2)));
        TB_TRY(cudaMemcpy(p->d_zap, p->zap.data(), p->zap.size() * sizeof(uint2), cudaMemcpyHostToDevice));
    }
#undef TB_TRY
    cufftHandle h;
    int rc = get_fft_plan(p, B, &h);
    if (rc) { destroy(p); return rc; }
    // series + fill value (+ whitening, which uses the chunk scratch allocated above)
    rc = load_series(p, series);
    if (rc) { destroy(p); return rc; }
    pin_series_in_l2(p);
    if (cudaStreamSynchronize(p->stream) != cudaSuccess) { destroy(p); return TB_ERR_CUDA; }
    *out = p;
    return TB_OK;
}

int tb_plan_set_series(tb_plan* p, const float* series)
{
    if (!p || !series) return fail(p, TB_ERR_INVALID_ARG, "null argument");
    TB_CUDA(p, cudaSetDevice(p->device));
    const int rc = load_series(p, series);
    return rc;
}

int tb_plan_destroy(tb_plan* plan)
{
    destroy(plan);
    return TB_OK;
}

int tb_plan_info(const tb_plan* plan, float* fill_value, uint32_t* chunk_templates, uint32_t* k_lo)
{
    if (!plan) return TB_ERR_INVALID_ARG;
    if (fill_value) *fill_value = plan->fill;
    if (chunk_templates) *chunk_templates = plan->chunk;
    if (k_lo) *k_lo = plan->k_lo;
    return TB_OK;
}

int tb_template_knot_log2(const tb_plan* plan, const tb_template* tmpl, int32_t* log2_h)
{
    if (!plan || !tmpl || !log2_h) return TB_ERR_INVALID_ARG;
    std::string why;
    if (validate_template(*tmpl, plan->tsamp, &why)) return TB_ERR_INVALID_ARG;
    TmplDev d;
    EllCoef ec;
    make_tmpl(*tmpl, plan->tsamp, &d, plan->ell ? &ec : nullptr);
    *log2_h = d.log2h;
    return TB_OK;
}

int tb_search_templates(tb_plan* p, const tb_template* tmpl, uint64_t n_templates, uint32_t first_template_id,
                        const uint32_t* folds, uint32_t n_folds, double sigma_threshold)
{
    if (!p) return TB_ERR_INVALID_ARG;
    if (n_templates && !tmpl) return fail(p, TB_ERR_INVALID_ARG, "tmpl is NULL");
    if (n_templates > 0xffffffffull - first_template_id) return fail(p, TB_ERR_INVALID_ARG, "template ids overflow 32 bits");
    FoldParams fp;
    int rc = make_fold_params(p, folds, n_folds, sigma_threshold, &fp);
    if (rc) return rc;
    TB_CUDA(p, cudaSetDevice(p->device));
    p->last = {};
    p->events_used = 0;
    p->last.n_templates = n_templates;
    p->last.n_samples = p->n;
    p->last.chunk_templates = p->chunk;
    p->last.model_bytes_per_template = 22ull * p->n;
    if (n_templates == 0) return TB_OK;
    TB_CUDA(p, cudaMemsetAsync(p->d_cursor + 1, 0, sizeof(unsigned long long), p->stream));
    rc = upload_templates(p, tmpl, n_templates);
    if (rc) return rc;

    // two runs of chunks: the templates the fused path takes (positions [0, n_own) of the staging
    // order), then the rest through k_resample + cuFFT; fft_path_used is the OR of the two
    p->last.fft_path_used = (p->n_own ? 2u : 0u) | (p->n_own < n_templates ? 1u : 0u);
    auto next_events = [&](EventSet** es) -> int {
        *es = nullptr;
        if (!p->timings) return TB_OK;
        if (p->events_used == p->events.size()) {
            EventSet ne;
            for (auto& e : ne.e) TB_CUDA(p, cudaEventCreate(&e));
            for (auto& e : ne.k) TB_CUDA(p, cudaEventCreate(&e));
            p->events.push_back(ne);
        }
        *es = &p->events[p->events_used++];
        (*es)->k_used = false;
        return TB_OK;
    };
    // K0 (+ the upload of the chunk's constants) on the side stream: queue it for chunk [off, off + nt)
    auto queue_k0 = [&](uint64_t off, uint32_t nt, EventSet* es, bool after_p1) -> int {
        if (int r = stage_chunk(p, tmpl, off, nt, first_template_id, p->s_k0)) return r;
        if (after_p1) TB_CUDA(p, cudaStreamWaitEvent(p->s_k0, p->ev_p1, 0));          // the segment table is free again
        if (es) { TB_CUDA(p, cudaEventRecord(es->k[0], p->s_k0)); es->k_used = true; }
        if (int r = run_k0(p, off, nt, p->s_k0)) return r;
        if (es) TB_CUDA(p, cudaEventRecord(es->k[1], p->s_k0));
        TB_CUDA(p, cudaEventRecord(p->ev_k0, p->s_k0));
        p->last.n_kernel_launches += 1;
        return TB_OK;
    };
    for (int part = 0; part < 2; ++part) {
        const bool own = part == 0;
        const uint64_t lo = own ? 0 : p->n_own, hi = own ? p->n_own : n_templates;
        EventSet *es = nullptr, *es_next = nullptr;
        if (own && lo < hi) {                            // everything queued so far (earlier calls read d_tmpl / d_seg) first
            TB_CUDA(p, cudaEventRecord(p->ev_main, p->stream));
            TB_CUDA(p, cudaStreamWaitEvent(p->s_k0, p->ev_main, 0));
            if ((rc = next_events(&es_next))) return rc;
            if ((rc = queue_k0(lo, (uint32_t)std::min<uint64_t>(p->chunk, hi - lo), es_next, false))) return rc;
        }
        for (uint64_t off = lo; off < hi; off += p->chunk) {
            const uint32_t nt = (uint32_t)std::min<uint64_t>(p->chunk, hi - off);
            if (own) {                                   // K0 (side stream) | P1 | P2 | transpose + unpack + spectrum + median + normalise
                es = es_next;
                es_next = nullptr;
                if (es) TB_CUDA(p, cudaEventRecord(es->e[0], p->stream));
                TB_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_k0, 0));
                if (es) TB_CUDA(p, cudaEventRecord(es->e[1], p->stream));
                if ((rc = run_p1(p, off, nt, nullptr, nullptr))) return rc;
                if (es) TB_CUDA(p, cudaEventRecord(es->e[2], p->stream));
                TB_CUDA(p, cudaEventRecord(p->ev_p1, p->stream));
                if (off + p->chunk < hi) {               // the next chunk's knots run under the rest of this chunk (measured: they
                                                         // fit beside the spectrum former's CTAs, not beside the harmonic summer's)
                    if ((rc = next_events(&es_next))) return rc;
                    if ((rc = queue_k0(off + p->chunk, (uint32_t)std::min<uint64_t>(p->chunk, hi - off - p->chunk), es_next, true))) return rc;
                }
                if ((rc = run_own_pass2(p, nt))) return rc;
                if (es) TB_CUDA(p, cudaEventRecord(es->e[3], p->stream));
                if ((rc = run_spectrum_t(p, nt))) return rc;
                p->last.n_kernel_launches += (p->log2m2 == 16) ? 3 : 2;
            } else {
                if ((rc = stage_chunk(p, tmpl, off, nt, first_template_id, p->stream))) return rc;
                if ((rc = next_events(&es))) return rc;
                if (es) TB_CUDA(p, cudaEventRecord(es->e[0], p->stream));
                if (es) TB_CUDA(p, cudaEventRecord(es->e[1], p->stream));
                if ((rc = run_resample(p, off, nt, nullptr))) return rc;
                if (es) TB_CUDA(p, cudaEventRecord(es->e[2], p->stream));
                if ((rc = run_fft(p, nt))) return rc;
                if (es) TB_CUDA(p, cudaEventRecord(es->e[3], p->stream));
                if ((rc = run_spectrum(p, nt, nullptr))) return rc;
                p->last.n_kernel_launches += 1;
            }
            if (es) TB_CUDA(p, cudaEventRecord(es->e[4], p->stream));
            if ((rc = run_hsum(p, off, nt, fp))) return rc;
            if (es) TB_CUDA(p, cudaEventRecord(es->e[5], p->stream));
            p->last.n_chunks++;
            p->last.n_kernel_launches += 2;
        }
    }
    return TB_OK;
}

int tb_get_timings(tb_plan* p, tb_timings* out)
{
    if (!p || !out) return TB_ERR_INVALID_ARG;
    TB_CUDA(p, cudaSetDevice(p->device));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    tb_timings t = p->last;
    {
        unsigned long long fb = 0;
        TB_CUDA(p, cudaMemcpy(&fb, p->d_cursor + 1, sizeof(fb), cudaMemcpyDeviceToHost));
        t.n_median_fallbacks = fb;
    }
    t.ms_delay = t.ms_resample = t.ms_fft = t.ms_spectrum = t.ms_normalise = t.ms_hsum = t.ms_total = 0.0;
    for (size_t i = 0; i < p->events_used; ++i) {
        float ms[5];
        for (int s = 0; s < 5; ++s) TB_CUDA(p, cudaEventElapsedTime(&ms[s], p->events[i].e[s], p->events[i].e[s + 1]));
        if (p->events[i].k_used) TB_CUDA(p, cudaEventElapsedTime(&ms[0], p->events[i].k[0], p->events[i].k[1]));   // K0 ran on the side stream
        t.ms_delay += ms[0]; t.ms_resample += ms[1]; t.ms_fft += ms[2]; t.ms_spectrum += ms[3]; t.ms_hsum += ms[4];
    }
    if (p->events_used) {
        float tot = 0.f;
        TB_CUDA(p, cudaEventElapsedTime(&tot, p->events[0].e[0], p->events[p->events_used - 1].e[5]));
        t.ms_total = tot;
    }
    *out = t;
    return TB_OK;
}

int tb_clear_candidates(tb_plan* p)
{
    if (!p) return TB_ERR_INVALID_ARG;
    TB_CUDA(p, cudaSetDevice(p->device));
    TB_CUDA(p, cudaMemsetAsync(p->d_cursor, 0, sizeof(unsigned long long), p->stream));
    return TB_OK;
}

int tb_get_candidates(tb_plan* p, tb_candidate* out, uint64_t capacity, uint64_t* n_total)
{
    if (!p || !n_total) return fail(p, TB_ERR_INVALID_ARG, "null argument");
    TB_CUDA(p, cudaSetDevice(p->device));
    unsigned long long count = 0;
    TB_CUDA(p, cudaMemcpyAsync(&count, p->d_cursor, sizeof(count), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    *n_total = count;
    const uint64_t stored = std::min<uint64_t>(count, p->max_cand);
    if (stored > 0 && (!out || capacity < stored)) return fail(p, TB_ERR_CAPACITY, "output buffer too small");
    if (stored > 0) {
        TB_CUDA(p, cudaMemcpyAsync(out, p->d_cand, stored * sizeof(Candidate), cudaMemcpyDeviceToHost, p->stream));
        TB_CUDA(p, cudaStreamSynchronize(p->stream));
        std::sort(out, out + stored, [](const tb_candidate& a, const tb_candidate& b) {
            if (a.template_id != b.template_id) return a.template_id < b.template_id;
            if (a.fold != b.fold) return a.fold < b.fold;
            return a.bin < b.bin;
        });
    }
    TB_CUDA(p, cudaMemsetAsync(p->d_cursor, 0, sizeof(unsigned long long), p->stream));
    if (count > p->max_cand) return fail(p, TB_ERR_OVERFLOW, "candidate buffer overflow: " + std::to_string(count));
    return TB_OK;
}

int tb_debug_resample_indices(tb_plan* p, const tb_template* tmpl, int64_t* idx_out)
{
    if (!idx_out) return fail(p, TB_ERR_INVALID_ARG, "null argument");
    int rc = single_template_stage(p, tmpl);
    if (rc) return rc;
    long long* d_idx = nullptr;
    TB_CUDA(p, cudaMalloc(&d_idx, p->n * sizeof(long long)));
    if (p->n_own) {
        float* d_y = nullptr;
        cudaError_t e = cudaMalloc(&d_y, p->n * sizeof(float));
        if (e != cudaSuccess) { cudaFree(d_idx); return fail(p, TB_ERR_NOMEM, "debug buffer"); }
        rc = run_own_pass1(p, 0, 1, d_idx, d_y);
        cudaStreamSynchronize(p->stream);
        cudaFree(d_y);
    } else
    rc = run_resample(p, 0, 1, d_idx);
    if (!rc) {
        cudaError_t e = cudaMemcpyAsync(idx_out, d_idx, p->n * sizeof(long long), cudaMemcpyDeviceToHost, p->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
        if (e != cudaSuccess) rc = fail(p, TB_ERR_CUDA, cudaGetErrorString(e));
    }
    cudaFree(d_idx);
    return rc;
}

int tb_debug_resampled(tb_plan* p, const tb_template* tmpl, float* y_out)
{
    if (!y_out) return fail(p, TB_ERR_INVALID_ARG, "null argument");
    int rc = single_template_stage(p, tmpl);
    if (rc) return rc;
    if (p->n_own) {
        long long* d_idx = nullptr;
        float* d_y = nullptr;
        TB_CUDA(p, cudaMalloc(&d_idx, p->n * sizeof(long long)));
        cudaError_t e = cudaMalloc(&d_y, p->n * sizeof(float));
        if (e != cudaSuccess) { cudaFree(d_idx); return fail(p, TB_ERR_NOMEM, "debug buffer"); }
        rc = run_own_pass1(p, 0, 1, d_idx, d_y);
        if (!rc) {
            e = cudaMemcpyAsync(y_out, d_y, p->n * sizeof(float), cudaMemcpyDeviceToHost, p->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
            if (e != cudaSuccess) rc = fail(p, TB_ERR_CUDA, cudaGetErrorString(e));
        }
        cudaStreamSynchronize(p->stream);
        cudaFree(d_idx); cudaFree(d_y);
        return rc;
    }
    if ((rc = run_resample(p, 0, 1, nullptr))) return rc;
    TB_CUDA(p, cudaMemcpyAsync(y_out, p->d_resampled, p->n * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    return TB_OK;
}

int tb_debug_spectrum(tb_plan* p, const tb_template* tmpl, float* p_interbinned, float* p_normalised, float* medians)
{
    int rc = single_template_stage(p, tmpl);
    if (rc) return rc;
    const bool own = p->n_own != 0;
    if (own) {
        if ((rc = run_own_pass1(p, 0, 1, nullptr, nullptr))) return rc;
        if ((rc = run_own_pass2(p, 1))) return rc;
    } else {
        if ((rc = run_resample(p, 0, 1, nullptr))) return rc;
        if ((rc = run_fft(p, 1))) return rc;
    }
    float* d_raw = nullptr;
    TB_CUDA(p, cudaMalloc(&d_raw, p->nsp * sizeof(float)));
    rc = own ? run_spectrum_t(p, 1, d_raw) : run_spectrum(p, 1, d_raw);
    cudaError_t e = cudaSuccess;
    if (!rc && p_interbinned) e = cudaMemcpyAsync(p_interbinned, d_raw, p->nsp * sizeof(float), cudaMemcpyDeviceToHost, p->stream);
    if (!rc && e == cudaSuccess && medians)
        e = cudaMemcpyAsync(medians, p->d_med, p->nblk * sizeof(float), cudaMemcpyDeviceToHost, p->stream);
    if (!rc && e == cudaSuccess && p_normalised)
        e = cudaMemcpyAsync(p_normalised, p->d_power, p->nsp * sizeof(float), cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    cudaFree(d_raw);
    if (rc) return rc;
    if (e != cudaSuccess) return fail(p, TB_ERR_CUDA, cudaGetErrorString(e));
    return TB_OK;
}

int tb_debug_series(tb_plan* p, float* x_out, double* kappa_out)
{
    if (!p) return TB_ERR_INVALID_ARG;
    TB_CUDA(p, cudaSetDevice(p->device));
    if (x_out) TB_CUDA(p, cudaMemcpyAsync(x_out, p->d_series, p->n * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    if (kappa_out) *kappa_out = p->whiten ? (double)p->kappa : 0.0;
    return TB_OK;
}

int tb_debug_hsums(tb_plan* p, const tb_template* tmpl, float* sums_out)
{
    if (!sums_out) return fail(p, TB_ERR_INVALID_ARG, "null argument");
    int rc = single_template_stage(p, tmpl);
    if (rc) return rc;
    if (p->n_own) {
        if ((rc = run_own_pass1(p, 0, 1, nullptr, nullptr))) return rc;
        if ((rc = run_own_pass2(p, 1))) return rc;
        if ((rc = run_spectrum_t(p, 1))) return rc;
    } else {
        if ((rc = run_resample(p, 0, 1, nullptr))) return rc;
        if ((rc = run_fft(p, 1))) return rc;
        if ((rc = run_spectrum(p, 1, nullptr))) return rc;
    }
    // the production harmonic summer with its tap on and thresholds at +inf (no candidate is emitted)
    FoldParams fp;
    for (int L = 0; L < 5; ++L) { fp.thr[L] = std::numeric_limits<float>::infinity(); fp.mu[L] = 0.f; fp.inv_s[L] = 0.f; fp.lo[L] = 0; }
    float* d_tap = nullptr;
    TB_CUDA(p, cudaMalloc(&d_tap, 5 * p->nsp * sizeof(float)));
    rc = run_hsum(p, 0, 1, fp, d_tap);
    cudaError_t e = cudaSuccess;
    if (!rc) e = cudaMemcpyAsync(sums_out, d_tap, 5 * p->nsp * sizeof(float), cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    cudaFree(d_tap);
    if (rc) return rc;
    if (e != cudaSuccess) return fail(p, TB_ERR_CUDA, cudaGetErrorString(e));
    return TB_OK;
}

}  // extern "C"

// ---- f1: candidate reduction (tb_reduce.cuh) --------------------------------------------------
namespace {

size_t sort_pad(size_t n)
{
    size_t p = BS_TILE;
    while (p < n) p <<= 1;
    return p;
}

// ascending bitonic sort of npad records (npad a power of two >= BS_TILE)
int device_sort(tb_plan* p, SortRec* r, size_t npad)
{
    k_bitonic_tiles<<<(unsigned)(npad / BS_TILE), BS_THREADS, 0, p->stream>>>(r);
    for (size_t size = 2 * (size_t)BS_TILE; size <= npad; size <<= 1) {
        for (size_t j = size >> 1; j >= (size_t)BS_TILE; j >>= 1)
            k_bitonic_step<<<(unsigned)((npad / 2 + 255) / 256), 256, 0, p->stream>>>(r, npad, size, j);
        k_bitonic_finish<<<(unsigned)(npad / BS_TILE), BS_THREADS, 0, p->stream>>>(r, size);
    }
    TB_CUDA(p, cudaGetLastError());
    return TB_OK;
}

unsigned blocks_for(size_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

extern "C" {

int tb_debug_set_candidates(tb_plan* p, const tb_candidate* cands, uint64_t n)
{
    if (!p || (n && !cands)) return fail(p, TB_ERR_INVALID_ARG, "null argument");
    if (n > p->max_cand) return fail(p, TB_ERR_CAPACITY, "more rows than max_candidates");
    for (uint64_t i = 0; i < n; ++i)
        if (cands[i].fold > TB_MAX_FOLD || cands[i].bin >= p->nsp) return fail(p, TB_ERR_INVALID_ARG, "row " + std::to_string(i) + ": fold or bin out of range");
    TB_CUDA(p, cudaSetDevice(p->device));
    const unsigned long long count = n;
    if (n) TB_CUDA(p, cudaMemcpyAsync(p->d_cand, cands, n * sizeof(Candidate), cudaMemcpyHostToDevice, p->stream));
    TB_CUDA(p, cudaMemcpyAsync(p->d_cursor, &count, sizeof(count), cudaMemcpyHostToDevice, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    return TB_OK;
}

int tb_reduce_candidates(tb_plan* p, double freq_tol_bins, tb_group* groups_out, uint64_t capacity, uint64_t* n_groups,
                         uint32_t* member_of, uint64_t member_capacity)
{
    if (!p || !n_groups) return fail(p, TB_ERR_INVALID_ARG, "null argument");
    if (!(freq_tol_bins >= 0) || freq_tol_bins > 1e6) return fail(p, TB_ERR_INVALID_ARG, "freq_tol_bins must be in [0, 1e6]");
    *n_groups = 0;
    TB_CUDA(p, cudaSetDevice(p->device));
    const int64_t tol16 = freq_tol_bins == 0.0 ? 16 : (int64_t)std::llround(16.0 * freq_tol_bins);
    unsigned long long count = 0;
    TB_CUDA(p, cudaMemcpyAsync(&count, p->d_cursor, sizeof(count), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    if (count > p->max_cand) return fail(p, TB_ERR_OVERFLOW, "candidate buffer overflow: " + std::to_string(count));
    const size_t n = (size_t)count;
    if (n == 0) return TB_OK;
    if (member_of && member_capacity < n) return fail(p, TB_ERR_CAPACITY, "member_of too small");

    DevBufs mem;
    SortRec *srt = nullptr, *rank = nullptr, *gt = nullptr;
    Peak* peaks = nullptr;
    uint32_t *peak_of = nullptr, *F = nullptr, *Fs = nullptr, *rank_at = nullptr, *rank_of_peak = nullptr, *gid = nullptr, *d_member = nullptr;
    int* state = nullptr;
    unsigned int* ctr = nullptr;                     // [0] peaks, [1] undecided, [2] groups
    Group* groups = nullptr;
    const size_t npad = sort_pad(n);
    TB_CUDA(p, mem.get(&srt, npad));
    TB_CUDA(p, mem.get(&peaks, n));
    TB_CUDA(p, mem.get(&peak_of, n));
    TB_CUDA(p, mem.get(&ctr, 4));
    TB_CUDA(p, cudaMemsetAsync(ctr, 0, 4 * sizeof(unsigned int), p->stream));

    // R1: sort by (template, fold, bin), runs of adjacent bins -> peaks
    k_red_det_keys<<<blocks_for(npad), 256, 0, p->stream>>>(p->d_cand, n, npad, srt);
    if (int rc = device_sort(p, srt, npad)) return rc;
    k_red_peaks<<<blocks_for(n), 256, 0, p->stream>>>(p->d_cand, srt, n, peaks, peak_of, ctr);
    unsigned int np = 0;
    TB_CUDA(p, cudaMemcpyAsync(&np, ctr, sizeof(np), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));

    // R2: rank by (sigma descending, template, fold, bin)
    const size_t ppad = sort_pad(np);
    TB_CUDA(p, mem.get(&rank, ppad));
    TB_CUDA(p, mem.get(&gt, ppad));
    TB_CUDA(p, mem.get(&F, np));
    TB_CUDA(p, mem.get(&Fs, np));
    TB_CUDA(p, mem.get(&rank_at, np));
    TB_CUDA(p, mem.get(&state, np));
    TB_CUDA(p, mem.get(&rank_of_peak, np));
    TB_CUDA(p, mem.get(&gid, np));
    TB_CUDA(p, mem.get(&groups, np));
    TB_CUDA(p, mem.get(&d_member, n));
    k_red_peak_keys<<<blocks_for(ppad), 256, 0, p->stream>>>(peaks, np, ppad, rank);
    if (int rc = device_sort(p, rank, ppad)) return rc;
    k_red_rank_init<<<blocks_for(np), 256, 0, p->stream>>>(peaks, rank, np, F, state, rank_of_peak);

    // the same peaks sorted by F (gt is free until R4): the windows of R3 are binary searches in Fs
    k_red_freq_keys<<<blocks_for(ppad), 256, 0, p->stream>>>(F, np, ppad, gt);
    if (int rc = device_sort(p, gt, ppad)) return rc;
    k_red_freq_split<<<blocks_for(np), 256, 0, p->stream>>>(gt, np, Fs, rank_at);

    // R3: rounds until every peak is a head or absorbed (each round decides at least the strongest open peak).
    // Four rounds are queued per look at the counter (most lists are done after two or three; a round
    // with nothing left to decide costs one read per peak), so the host synchronises once per batch.
    constexpr int ROUNDS_PER_CHECK = 4;
    for (size_t round = 0; round <= np; round += ROUNDS_PER_CHECK) {
        TB_CUDA(p, cudaMemsetAsync(ctr + 1, 0, sizeof(unsigned int), p->stream));
        for (int k = 0; k < ROUNDS_PER_CHECK; ++k)
            k_red_distill_round<<<blocks_for(np), 256, 0, p->stream>>>(F, Fs, rank_at, state, np, tol16,
                                                                       k == ROUNDS_PER_CHECK - 1 ? ctr + 1 : nullptr);
        unsigned int open = 0;
        TB_CUDA(p, cudaMemcpyAsync(&open, ctr + 1, sizeof(open), cudaMemcpyDeviceToHost, p->stream));
        TB_CUDA(p, cudaStreamSynchronize(p->stream));
        if (open == 0) break;
    }

    // R4: number the heads, fill the group records, count distinct templates, map detections to groups
    k_red_number_heads<<<1, 1024, 0, p->stream>>>(state, np, gid, ctr + 2);
    TB_CUDA(p, cudaMemsetAsync(groups, 0, (size_t)np * sizeof(Group), p->stream));
    k_red_groups<<<blocks_for(ppad), 256, 0, p->stream>>>(peaks, rank, state, gid, np, ppad, groups, gt);
    if (int rc = device_sort(p, gt, ppad)) return rc;
    k_red_count_templates<<<blocks_for(np), 256, 0, p->stream>>>(gt, np, groups);
    k_red_members<<<blocks_for(n), 256, 0, p->stream>>>(peak_of, rank_of_peak, state, gid, n, d_member);
    TB_CUDA(p, cudaGetLastError());
    unsigned int ng = 0;
    TB_CUDA(p, cudaMemcpyAsync(&ng, ctr + 2, sizeof(ng), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    *n_groups = ng;
    if (!groups_out || capacity < ng) return fail(p, TB_ERR_CAPACITY, "groups_out too small");
    TB_CUDA(p, cudaMemcpyAsync(groups_out, groups, (size_t)ng * sizeof(Group), cudaMemcpyDeviceToHost, p->stream));
    if (member_of) TB_CUDA(p, cudaMemcpyAsync(member_of, d_member, n * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
    TB_CUDA(p, cudaStreamSynchronize(p->stream));
    return TB_OK;
}

}  // extern "C"
