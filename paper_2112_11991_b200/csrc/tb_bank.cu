// tb_bank.cu -- random template-bank generator on the device (include/tb.h
// "template bank" section).  PAPER.md sections 2.2-2.7:
//   density  rho(lambda) = sqrt|det gamma|, gamma = frequency-projected metric (eq 13, eq 14
//            L101, eq 22) of the phase model eq 1-2 (L35-41) with the e-series of eqs 15-16
//            (L106-111, App. B); circular: eq 4 (L49)
//   box      Table 1 (L196-216) with eq 31 (L248)
//   placement: accept proposal i iff u_i5 rho_max < rho(lambda_i) (L263, reading G28), kept in order
//
// How the determinant is formed (differs from the oracle's literal eq 13 -> eq 22 -> det on purpose):
// gamma is the Gram matrix of the derivative functions d_a Phi(t) after the constant and d_f Phi have
// been projected out, under the inner product <u v>_T.  One CTA samples the n_par + 1 functions at
// 1024 (or 4096) Gauss-Legendre nodes, orthogonalises the columns (1, d_f, d_1, ..., d_n) by modified
// Gram-Schmidt with block-wide fp64 dot products, and sqrt(det gamma) = prod_{a >= 1} |r_a| of the
// residual norms.  For P_orb >> T the metric has a condition number of 1e11 and a plain fp64
// evaluation of eq 13 loses every digit to cancellation; this route loses sqrt(cond) ~ 3e5 of 1e16.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <vector>

#include "../../include/tb.h"

namespace tbbank {

constexpr int GL = 32;                        // Gauss-Legendre points per panel
constexpr int NPT = 8;                        // nodes per thread
constexpr int MAXP = 6;                       // columns: f + up to 5 orbital parameters (the constant is implicit)
constexpr double TWO_PI = 6.283185307179586476925286766559;

struct Space {                                // tb_bank_space, digested on the host
    double t_obs, f0, p_min, p_span, k_tau, e_max;   // k_tau: tau_max = k_tau Omega^(-2/3) (eq 31)
    int elliptical, n_par;                    // n_par = 3 or 5 orbital parameters
};

__constant__ double c_glx[GL], c_glw[GL];     // nodes in (-1, 1), weights summing to 2
__constant__ double c_C[8][7], c_S[8][7];     // coefficient of e^p in C_k, S_k (App. B), p = 0..6

// C_k(e), S_k(e) and d/de by Horner over the printed table: thread k < 8 fills ser[0..3][k]
__device__ __forceinline__ void series_coeffs(double e, double (*ser)[8])
{
    if (threadIdx.x < 8) {
        const int k = threadIdx.x;
        double c = 0, s = 0, dc = 0, ds = 0;
        for (int p = 6; p >= 0; --p) {
            dc = dc * e + c; ds = ds * e + s;
            c = c * e + c_C[k][p]; s = s * e + c_S[k][p];
        }
        ser[0][k] = c; ser[1][k] = s; ser[2][k] = dc; ser[3][k] = ds;
    }
    __syncthreads();
}

// block-wide sum in a fixed order (deterministic): lanes by shuffle tree, then the warps in order
__device__ __forceinline__ double block_sum(double v, double* s_red)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    __syncthreads();                          // s_red free again
    if ((threadIdx.x & 31) == 0) s_red[w] = v;
    __syncthreads();
    double t = 0;
    for (int i = 0; i < nw; ++i) t += s_red[i];
    return t;
}

// rho = sqrt|det gamma| at lam = (tau, Omega, alpha, psi, e); blockDim.x * NPT quadrature nodes
__device__ double density_cta(const Space& sp, double tau, double om, double al, double psi, double e, double* s_red,
                              double (*ser)[8])
{
    const int n_col = sp.n_par + 1;           // f, then the orbital parameters
    double col[MAXP][NPT], w[NPT];
    const double *C = ser[0], *S = ser[1], *dC = ser[2], *dS = ser[3];
    if (sp.elliptical) series_coeffs(e, ser);
    double sps, cps;
    sincos(psi, &sps, &cps);
    const int panels = (blockDim.x * NPT) / GL;
    const double hw = 0.5 * sp.t_obs / (double)panels;           // half width of a panel
    const double kf = TWO_PI * sp.f0;
#pragma unroll
    for (int j = 0; j < NPT; ++j) {
        const int node = threadIdx.x * NPT + j;
        const int pan = node / GL, q = node % GL;
        const double t = hw * ((double)(2 * pan + 1) + c_glx[q]);
        w[j] = c_glw[q] * (0.5 / (double)panels);                // weights sum to 1 (eq 14)
        double s1, c1;
        sincos(om * t + al, &s1, &c1);
        double X, XM, Xp = 0, Xe = 0;
        if (sp.elliptical) {
            double cc = C[0], ss = 0, ccM = 0, ssM = 0, cce = dC[0], sse = 0;
            double ck = 1.0, sk = 0.0;
#pragma unroll
            for (int k = 1; k < 8; ++k) {                        // (cos kM, sin kM) by rotation
                const double cn = ck * c1 - sk * s1, sn = sk * c1 + ck * s1;
                ck = cn; sk = sn;
                cc += C[k] * ck;  ss += S[k] * sk;
                ccM -= (double)k * C[k] * sk;  ssM += (double)k * S[k] * ck;
                cce += dC[k] * ck;  sse += dS[k] * sk;
            }
            X = sps * cc + cps * ss;  XM = sps * ccM + cps * ssM;
            Xp = cps * cc - sps * ss; Xe = sps * cce + cps * sse;
        } else {
            X = s1; XM = c1;
        }
        col[0][j] = TWO_PI * (t + tau * X);                      // d/d f0   (reading G27: with the tau X term)
        col[1][j] = kf * X;                                      // d/d tau
        col[2][j] = kf * tau * t * XM;                           // d/d Omega
        col[3][j] = kf * tau * XM;                               // d/d alpha
        col[4][j] = kf * tau * Xp;                               // d/d psi
        col[5][j] = kf * tau * Xe;                               // d/d e
    }
    // modified Gram-Schmidt: remove the constant (the mean, eq 13's second term), then column by column
    double rho = 1.0;
#pragma unroll
    for (int a = 0; a < MAXP; ++a) {
        if (a >= n_col) break;
        double m = 0;
#pragma unroll
        for (int j = 0; j < NPT; ++j) m += w[j] * col[a][j];
        m = block_sum(m, s_red);
#pragma unroll
        for (int j = 0; j < NPT; ++j) col[a][j] -= m;
#pragma unroll
        for (int b = 0; b < MAXP; ++b) {
            if (b >= a) break;
            double d = 0;                                         // col[b] is already normalised
#pragma unroll
            for (int j = 0; j < NPT; ++j) d += w[j] * col[b][j] * col[a][j];
            d = block_sum(d, s_red);
#pragma unroll
            for (int j = 0; j < NPT; ++j) col[a][j] -= d * col[b][j];
        }
        double nn = 0;
#pragma unroll
        for (int j = 0; j < NPT; ++j) nn += w[j] * col[a][j] * col[a][j];
        nn = block_sum(nn, s_red);
        const double nrm = sqrt(nn);
        if (a > 0) rho *= nrm;                                   // eq 22: the f column is projected out, not counted
        const double inv = nrm > 0 ? 1.0 / nrm : 0.0;
#pragma unroll
        for (int j = 0; j < NPT; ++j) col[a][j] *= inv;
    }
    return rho;
}

// proposal of Table 1 from six uniforms (oracle/tb_bank.py::proposal states the same map)
__device__ __forceinline__ void propose(const Space& sp, const double* __restrict__ u, double (&lam)[5], double& q)
{
    const double p = sp.p_min + u[0] * sp.p_span;
    const double om = TWO_PI / p;
    const double tmax = sp.k_tau / cbrt(om * om);                // eq 31
    lam[0] = u[1] * tmax; lam[1] = om; lam[2] = TWO_PI * u[2];
    lam[3] = sp.elliptical ? TWO_PI * u[3] : 0.0;
    lam[4] = sp.elliptical ? u[4] * sp.e_max : 0.0;
    q = (p * p / TWO_PI) / sp.p_span / tmax / TWO_PI;            // pdf of the proposal in (tau, Omega, alpha[, psi, e])
    if (sp.elliptical) q /= TWO_PI * sp.e_max;
}

// one CTA per point.  MODE 0: lam given ([n][5]); MODE 1: uniforms given ([n][6]) -> rho, accept flag, rho / q
template <int MODE>
__global__ void __launch_bounds__(512)
k_bank_density(Space sp, const double* __restrict__ in, double rho_max, double* __restrict__ rho_out,
               unsigned char* __restrict__ accept, double* __restrict__ rho_over_q)
{
    __shared__ double s_red[16];
    __shared__ double s_ser[4][8];
    const size_t i = blockIdx.x;
    double lam[5], q = 1.0;
    if (MODE == 0) {
#pragma unroll
        for (int k = 0; k < 5; ++k) lam[k] = in[i * 5 + k];
    } else {
        propose(sp, in + i * 6, lam, q);
    }
    const double rho = density_cta(sp, lam[0], lam[1], lam[2], lam[3], lam[4], s_red, s_ser);
    if (threadIdx.x == 0) {
        rho_out[i] = rho;
        if (MODE == 1) {
            accept[i] = (in[i * 6 + 5] * rho_max < rho) ? 1 : 0;
            rho_over_q[i] = rho / q;
        }
    }
}

// ordered compaction of the accepted proposals.  One CTA of 1024 threads walks the flags in order
// (the list is at most a few million entries and this is 1 byte per entry): running offset in a
// register, ballot + popc inside a warp, a 32-entry scan across the warps.  Also the volume sum.
__global__ void __launch_bounds__(1024)
k_bank_compact(Space sp, const double* __restrict__ uniforms, const unsigned char* __restrict__ accept,
               const double* __restrict__ rho_over_q, size_t n, tb_template* __restrict__ out, size_t capacity,
               unsigned long long* __restrict__ n_accepted, double* __restrict__ volume)
{
    __shared__ unsigned int s_cnt[32];
    __shared__ double s_sum[32];
    __shared__ unsigned long long s_base;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_base = 0;
    double vsum = 0.0;                                             // fixed order per thread, then a fixed tree
    __syncthreads();
    for (size_t i0 = 0; i0 < n; i0 += 1024) {
        const size_t i = i0 + threadIdx.x;
        const bool acc = i < n && accept[i];
        if (i < n) vsum += rho_over_q[i];
        const unsigned bal = __ballot_sync(0xffffffffu, acc);
        if (lane == 0) s_cnt[wid] = __popc(bal);
        __syncthreads();
        unsigned before = 0, total = 0;
        for (int w2 = 0; w2 < 32; ++w2) { const unsigned c = s_cnt[w2]; if (w2 < wid) before += c; total += c; }
        const unsigned long long pos = s_base + before + __popc(bal & ((1u << lane) - 1));
        if (acc && pos < capacity) {
            double lam[5], q;
            propose(sp, uniforms + i * 6, lam, q);
            tb_template t;
            t.p_orb_s = TWO_PI / lam[1]; t.tau_lts = lam[0]; t.phi0_rad = lam[2]; t.ecc = lam[4]; t.omega_rad = lam[3];
            out[pos] = t;
        }
        __syncthreads();
        if (threadIdx.x == 0) s_base += total;
        __syncthreads();
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vsum += __shfl_xor_sync(0xffffffffu, vsum, o);
    if (lane == 0) s_sum[wid] = vsum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0;
        for (int w2 = 0; w2 < 32; ++w2) t += s_sum[w2];
        *volume = n ? t / (double)n : 0.0;
        *n_accepted = s_base;
    }
}

}  // namespace tbbank

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
namespace {

using namespace tbbank;

// Appendix B of the paper, typed in here independently of the oracle's table:
// {k, power of e, numerator, denominator}
struct Term { int k, pw; long long num, den; };
const Term APP_B_C[] = {{0, 1, -1, 2}, {1, 0, 1, 1}, {1, 2, -3, 8}, {1, 4, 5, 192}, {1, 6, -7, 9216}, {2, 1, 1, 2}, {2, 3, -1, 3},
                        {2, 5, 1, 16}, {3, 2, 3, 8}, {3, 4, -45, 128}, {3, 6, 567, 5120}, {4, 3, 1, 3}, {4, 5, -2, 5},
                        {5, 4, 125, 384}, {5, 6, -4375, 9216}, {6, 5, 27, 80}, {7, 6, 16807, 46080}};
const Term APP_B_S[] = {{1, 0, 1, 1}, {1, 2, -5, 8}, {1, 4, -11, 192}, {1, 6, -457, 9216}, {2, 1, 1, 2}, {2, 3, -5, 12},
                        {2, 5, 1, 24}, {3, 2, 3, 8}, {3, 4, -51, 128}, {3, 6, 543, 5120}, {4, 3, 1, 3}, {4, 5, -13, 30},
                        {5, 4, 125, 384}, {5, 6, -4625, 9216}, {6, 5, 27, 80}, {7, 6, 16807, 46080}};

// 32-point Gauss-Legendre rule on (-1, 1): Newton on P_32 in long double from the Chebyshev guess
void gauss_legendre(double* x, double* w)
{
    const long double pi = 4.0L * atanl(1.0L);
    for (int i = 0; i < GL; ++i) {
        long double z = cosl(pi * (i + 0.75L) / (GL + 0.5L)), dp = 0;
        for (int it = 0; it < 100; ++it) {
            long double p0 = 1, p1 = z;
            for (int k = 2; k <= GL; ++k) { const long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
            dp = GL * (z * p1 - p0) / (z * z - 1);
            const long double dz = p1 / dp;
            z -= dz;
            if (fabsl(dz) < 1e-19L) break;
        }
        long double p0 = 1, p1 = z;
        for (int k = 2; k <= GL; ++k) { const long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
        dp = GL * (z * p1 - p0) / (z * z - 1);
        x[GL - 1 - i] = (double)z;
        w[GL - 1 - i] = (double)(2.0L / ((1 - z * z) * dp * dp));
    }
}

struct Dev {                                  // frees on scope exit
    std::vector<void*> p;
    ~Dev() { for (void* q : p) cudaFree(q); }
    template <class T> cudaError_t get(T** out, size_t n)
    {
        void* q = nullptr;
        cudaError_t e = cudaMalloc(&q, (n ? n : 1) * sizeof(T));
        if (e == cudaSuccess) { p.push_back(q); *out = static_cast<T*>(q); }
        return e;
    }
};

#define BK_CUDA(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { cudaGetLastError(); return e_ == cudaErrorMemoryAllocation ? TB_ERR_NOMEM : TB_ERR_CUDA; } } while (0)

constexpr double T_SUN_S = 4.925490947e-6;    // G M_sun / c^3, seconds

int digest(const tb_bank_space* s, Space* sp)
{
    if (!s || s->struct_size != sizeof(tb_bank_space)) return TB_ERR_INVALID_ARG;
    auto pos = [](double v) { return std::isfinite(v) && v > 0; };
    if (!pos(s->t_obs_s) || !pos(s->f_max_hz) || !pos(s->p_orb_min_s) || !(s->p_orb_max_s >= s->p_orb_min_s) ||
        !std::isfinite(s->p_orb_max_s) || !pos(s->m_comp_max) || !(s->m_pulsar_min >= 0) || !std::isfinite(s->m_pulsar_min) ||
        !(s->theta > 0 && s->theta <= 1) || (s->elliptical && !(s->e_max > 0 && s->e_max <= 0.3)))
        return TB_ERR_INVALID_ARG;
    sp->t_obs = s->t_obs_s; sp->f0 = s->f_max_hz; sp->p_min = s->p_orb_min_s; sp->p_span = s->p_orb_max_s - s->p_orb_min_s;
    sp->k_tau = (double)((long double)s->theta * cbrtl((long double)T_SUN_S) * (long double)s->m_comp_max /
                         cbrtl(powl((long double)s->m_pulsar_min + (long double)s->m_comp_max, 2.0L)));
    sp->e_max = s->e_max; sp->elliptical = s->elliptical ? 1 : 0; sp->n_par = s->elliptical ? 5 : 3;
    return TB_OK;
}

// quadrature size: 32-point panels must stay short against the 14th harmonic of the orbit
int threads_for(double orbits)
{
    if (!(orbits >= 0) || orbits > 28.0) return 0;
    return orbits <= 7.0 ? 128 : 512;         // 1024 or 4096 nodes
}

int upload_tables(int device)
{
    BK_CUDA(cudaSetDevice(device));
    double x[GL], w[GL], C[8][7] = {}, S[8][7] = {};
    gauss_legendre(x, w);
    for (const Term& t : APP_B_C) C[t.k][t.pw] = (double)((long double)t.num / (long double)t.den);
    for (const Term& t : APP_B_S) S[t.k][t.pw] = (double)((long double)t.num / (long double)t.den);
    BK_CUDA(cudaMemcpyToSymbol(c_glx, x, sizeof(x)));
    BK_CUDA(cudaMemcpyToSymbol(c_glw, w, sizeof(w)));
    BK_CUDA(cudaMemcpyToSymbol(c_C, C, sizeof(C)));
    BK_CUDA(cudaMemcpyToSymbol(c_S, S, sizeof(S)));
    return TB_OK;
}

}  // namespace

extern "C" {

int tb_bank_density(const tb_bank_space* space, const double* lam, uint64_t n, double* rho_out)
{
    Space sp;
    if (int rc = digest(space, &sp)) return rc;
    if ((!lam || !rho_out) && n) return TB_ERR_INVALID_ARG;
    if (n == 0) return TB_OK;
    if (n > 0x7fffffffull) return TB_ERR_INVALID_ARG;
    double orbits = 0;
    for (uint64_t i = 0; i < n; ++i) {
        const double* l = lam + 5 * i;
        for (int k = 0; k < 5; ++k) if (!std::isfinite(l[k])) return TB_ERR_INVALID_ARG;
        if (l[0] < 0 || !(l[1] > 0) || (sp.elliptical && (l[4] < 0 || l[4] > 0.3))) return TB_ERR_INVALID_ARG;   // psi, e are ignored when circular
        orbits = std::max(orbits, l[1] * sp.t_obs / TWO_PI);
    }
    const int threads = threads_for(orbits);
    if (!threads) return TB_ERR_INVALID_ARG;
    if (int rc = upload_tables(space->device)) return rc;
    Dev mem;
    double *d_in = nullptr, *d_rho = nullptr;
    BK_CUDA(mem.get(&d_in, 5 * n));
    BK_CUDA(mem.get(&d_rho, n));
    BK_CUDA(cudaMemcpy(d_in, lam, 5 * n * sizeof(double), cudaMemcpyHostToDevice));
    k_bank_density<0><<<(unsigned)n, threads>>>(sp, d_in, 0.0, d_rho, nullptr, nullptr);
    BK_CUDA(cudaGetLastError());
    BK_CUDA(cudaMemcpy(rho_out, d_rho, n * sizeof(double), cudaMemcpyDeviceToHost));
    return TB_OK;
}

int tb_bank_generate(const tb_bank_space* space, const double* uniforms, uint64_t n, double rho_max, tb_template* out,
                     uint64_t capacity, uint64_t* n_accepted, double* rho_out, double* volume_out)
{
    Space sp;
    if (int rc = digest(space, &sp)) return rc;
    if (!n_accepted || (!uniforms && n) || !(rho_max > 0) || !std::isfinite(rho_max)) return TB_ERR_INVALID_ARG;
    *n_accepted = 0;
    if (volume_out) *volume_out = 0.0;
    if (n == 0) return TB_OK;
    if (n > 0x7fffffffull) return TB_ERR_INVALID_ARG;
    for (uint64_t i = 0; i < 6 * n; ++i) if (!(uniforms[i] >= 0.0 && uniforms[i] < 1.0)) return TB_ERR_INVALID_ARG;
    const int threads = threads_for(sp.t_obs / sp.p_min);
    if (!threads) return TB_ERR_INVALID_ARG;
    if (int rc = upload_tables(space->device)) return rc;
    Dev mem;
    double *d_u = nullptr, *d_rho = nullptr, *d_roq = nullptr, *d_vol = nullptr;
    unsigned char* d_acc = nullptr;
    tb_template* d_out = nullptr;
    unsigned long long* d_n = nullptr;
    BK_CUDA(mem.get(&d_u, 6 * n));
    BK_CUDA(mem.get(&d_rho, n));
    BK_CUDA(mem.get(&d_roq, n));
    BK_CUDA(mem.get(&d_acc, n));
    BK_CUDA(mem.get(&d_out, capacity));
    BK_CUDA(mem.get(&d_n, 1));
    BK_CUDA(mem.get(&d_vol, 1));
    BK_CUDA(cudaMemcpy(d_u, uniforms, 6 * n * sizeof(double), cudaMemcpyHostToDevice));
    k_bank_density<1><<<(unsigned)n, threads>>>(sp, d_u, rho_max, d_rho, d_acc, d_roq);
    BK_CUDA(cudaGetLastError());
    k_bank_compact<<<1, 1024>>>(sp, d_u, d_acc, d_roq, (size_t)n, d_out, (size_t)capacity, d_n, d_vol);
    BK_CUDA(cudaGetLastError());
    unsigned long long na = 0;
    BK_CUDA(cudaMemcpy(&na, d_n, sizeof(na), cudaMemcpyDeviceToHost));
    *n_accepted = na;
    if (volume_out) BK_CUDA(cudaMemcpy(volume_out, d_vol, sizeof(double), cudaMemcpyDeviceToHost));
    if (rho_out) BK_CUDA(cudaMemcpy(rho_out, d_rho, n * sizeof(double), cudaMemcpyDeviceToHost));
    if (na > capacity || (na && !out)) return TB_ERR_CAPACITY;
    if (na) BK_CUDA(cudaMemcpy(out, d_out, na * sizeof(tb_template), cudaMemcpyDeviceToHost));
    return TB_OK;
}

int tb_bank_n_templates(double eta, double m_star, uint32_t n_dim, double volume, int32_t exact, double* n_out)
{
    if (!n_out || !(eta > 0 && eta < 1) || !(m_star > 0 && m_star <= 1) || n_dim < 1 || n_dim > 16 || !(volume > 0)) return TB_ERR_INVALID_ARG;
    const double cn = std::pow(3.14159265358979323846, 0.5 * n_dim) / std::tgamma(0.5 * n_dim + 1.0);     // eq 18
    const double x = std::pow(m_star, 0.5 * n_dim) * cn / volume;
    if (exact && !(x < 1)) return TB_ERR_INVALID_ARG;
    *n_out = exact ? std::log(1.0 - eta) / std::log1p(-x) : std::log(1.0 / (1.0 - eta)) / x;               // eq 20 / eq 21
    return TB_OK;
}

}  // extern "C"
