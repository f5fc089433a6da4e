// loc_solve.cu -- per-cell statistical-equilibrium solve: three kernels for the same
// equations.  k_solve_f: float32 in registers, the one that runs for species of up to LOC_SOLVE_F_MAXNL levels;
// k_solve_s: float64 with the matrix in shared memory (up to 16 levels, and species the register kernel does not take);
// k_solve: float64 with the matrix in local memory (any level count).
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "loc_internal.cuh"

// Statistical equilibrium of one cell per thread (DESIGN 5.5).  The rate matrix is a
// continuous-time Markov generator; its stationary vector is found with the subtraction-free GTH elimination
// in double precision (the oracle uses pivoted Gaussian elimination on the same equations).
template <int NLMAX>
__global__ void __launch_bounds__(128) k_solve(int64_t n, SpeciesDev sp, Selection S, const float *density, const float *tkin,
                                               const float *abundance, const float2 *cnt, float *pops, float2 *coef,
                                               unsigned int *maxrel_bits, const int32_t *child, int ali)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    bool act = i < n;
    if (act && child && child[i] >= 0) act = false;  // refined cell: no gas of its own
    float rel = 0.0f;
    if (act) {
        const int NL = sp.nlevel;
        double R[NLMAX * NLMAX];
        for (int k = 0; k < NL * NL; k++) R[k] = 0.0;
        double dens = density[i], T = tkin[i];
        double ntot = dens * (double)abundance[i];
        // radiative rates
        for (int t = 0; t < sp.ntrans; t++) {
            int u = sp.upper[t], l = sp.lower[t];
            double gr = sp.g[u] / sp.g[l];
            double sj = sp.bgocc[t], esc = 1.0;  // DESIGN R23: untraced transitions see the background only
            for (int k = 0; k < S.nsel; k++)
                if (S.sel[k] == t) {
                    float2 c = cnt[i * S.nsp + k];
                    sj = c.x;
                    esc = c.y;
                    if (!ali) {
                        // plain lambda iteration ("possible to run LOC without ALI"): the self term of
                        // Eq. 2 goes back into the radiation field and A_ul stays unscaled.  Step by step it equals
                        // (1 - ESC) times the source function of the populations the rays were traced with, whose
                        // occupation number is em / kap of the cell's coefficient record (DESIGN 5.2, 6.2)
                        float2 ke = coef[i * S.nsp + k];
                        if (ke.x != 0.0f) sj += (1.0 - esc) * ((double)ke.y / (double)ke.x);
                        esc = 1.0;
                    }
                }
            double Slu = gr * sp.A[t] * sj;  // = B_lu * Jbar
            R[u * NL + l] += sp.A[t] * esc + Slu / gr;
            R[l * NL + u] += Slu;
        }
        // collisions: linear interpolation in T, clamped; upward by detailed balance
        int j = 0;
        double f = 0.0;
        if (sp.ntemp > 1) {
            if (T <= sp.temps[0]) {
                j = 0;
                f = 0.0;
            } else if (T >= sp.temps[sp.ntemp - 1]) {
                j = sp.ntemp - 2;
                f = 1.0;
            } else {
                while (T > sp.temps[j + 1]) j++;
                f = (T - sp.temps[j]) / (sp.temps[j + 1] - sp.temps[j]);
            }
        }
        // Boltzmann factors g_k exp(-(E_k - E_0) / T) once per level (one exp per level instead of one per collisional pair)
        double bz[NLMAX];
        for (int k = 0; k < NL; k++) bz[k] = sp.g[k] * exp(-(sp.energy_K[k] - sp.energy_K[0]) / T);
        for (int k = 0; k < sp.ncoll; k++) {
            int u = sp.cu[k], l = sp.cl[k];
            double gd = sp.rates[(int64_t)j * sp.ncoll + k];
            if (sp.ntemp > 1) gd = (1.0 - f) * gd + f * sp.rates[(int64_t)(j + 1) * sp.ncoll + k];
            double gu = gd * bz[u] / bz[l];
            R[u * NL + l] += dens * gd;
            R[l * NL + u] += dens * gu;
        }
        // GTH elimination
        for (int q = NL - 1; q >= 1; q--) {
            double s = 0.0;
            for (int c = 0; c < q; c++) s += R[q * NL + c];
            double inv = s > 0.0 ? 1.0 / s : 0.0;
            for (int r = 0; r < q; r++) R[r * NL + q] *= inv;
            for (int r = 0; r < q; r++) {
                double rq = R[r * NL + q];
                for (int c = 0; c < q; c++)
                    if (c != r) R[r * NL + c] += rq * R[q * NL + c];
            }
        }
        double x[NLMAX];
        x[0] = 1.0;
        double tot = 1.0;
        for (int q = 1; q < NL; q++) {
            double s = 0.0;
            for (int r = 0; r < q; r++) s += x[r] * R[r * NL + q];
            x[q] = s;
            tot += s;
        }
        double sc = ntot / tot;
        for (int l = 0; l < NL; l++) {
            double nw = x[l] * sc;
            double old = pops[(int64_t)l * n + i];
            if (ntot > 0.0 && (nw >= 1e-10 * ntot || old >= 1e-10 * ntot))
                rel = fmaxf(rel, (float)(fabs(nw - old) / fmax(nw, 1e-300)));
            if (!isfinite(nw)) rel = INFINITY;  // reported by fetch_maxrel as LOC_ENONFINITE, never as "converged"
            x[l] = nw;
            pops[(int64_t)l * n + i] = (float)nw;
        }
        // refresh the line coefficients of the traced transitions from the unrounded solution
        for (int k = 0; k < S.nsp; k++) {
            float2 v = make_float2(0.f, 0.f);
            if (k < S.nsel) {
                v.x = (float)(S.ck[k] * (x[S.lower[k]] * (double)S.gratio[k] - x[S.upper[k]]));
                v.y = (float)(S.ck[k] * x[S.upper[k]]);
            }
            coef[i * S.nsp + k] = v;
        }
    }
    for (int o = 16; o >= 1; o >>= 1) rel = fmaxf(rel, __shfl_xor_sync(0xffffffffu, rel, o));
    if ((threadIdx.x & 31) == 0 && rel > 0.0f) atomicMax(maxrel_bits, __float_as_uint(rel));
}

// k_solve_s: the same equations and the same GTH elimination as k_solve, laid out for the SM instead of for the
// compiler's local-memory stack (profiles/r1_solve.md: k_solve<10> keeps R in 960 B of local memory per thread, 1.1 MB per
// SM at its occupancy -- the L1 hit rate is 60 % and 34 of 35 issue slots wait on the long scoreboard).  Here the rate
// matrix of a thread is a column of a shared-memory array R[NL*NL][threads] of doubles (conflict free, never leaves the
// SM), the species tables are staged in shared memory once per block, and NL is a compile-time constant for the common
// level counts (NLX > 0), so that the elimination is fully unrolled with static addresses and x[], bz[] are registers.
#define LOC_SOLVE_THREADS 32  // cells per block: 31 KB of matrices at 10 levels, 7 blocks per SM (64: 62 KB, 3 blocks = 6 warps; C3 1.50 -> 1.35 ms)
struct SolveTabs {   // byte offsets into the block's shared memory, after R
    int g, energy, A, bg, gr, upper, lower, cu, cl, temps, rates, bytes;
};

template <int NLX>
__global__ void __launch_bounds__(LOC_SOLVE_THREADS) k_solve_s(int64_t n, SpeciesDev sp, Selection S, const float *density, const float *tkin,
                                                               const float *abundance, const float2 *cnt, float *pops, float2 *coef,
                                                               unsigned int *maxrel_bits, const int32_t *child, int ali, SolveTabs TB)
{
    constexpr int NLM = NLX > 0 ? NLX : 16;
    extern __shared__ __align__(16) unsigned char s_raw[];
    const int NL = NLX > 0 ? NLX : sp.nlevel;
    const int tid = threadIdx.x;
    double *Rs = reinterpret_cast<double *>(s_raw);
    unsigned char *tb = s_raw + sizeof(double) * (NL * NL + 2 * NL) * LOC_SOLVE_THREADS;
    double *t_g = reinterpret_cast<double *>(tb + TB.g), *t_e = reinterpret_cast<double *>(tb + TB.energy);
    double *t_A = reinterpret_cast<double *>(tb + TB.A), *t_bg = reinterpret_cast<double *>(tb + TB.bg), *t_gr = reinterpret_cast<double *>(tb + TB.gr);
    double *t_temps = reinterpret_cast<double *>(tb + TB.temps), *t_rates = reinterpret_cast<double *>(tb + TB.rates);
    int *t_up = reinterpret_cast<int *>(tb + TB.upper), *t_lo = reinterpret_cast<int *>(tb + TB.lower);
    int *t_cu = reinterpret_cast<int *>(tb + TB.cu), *t_cl = reinterpret_cast<int *>(tb + TB.cl);
    for (int k = tid; k < NL; k += LOC_SOLVE_THREADS) {
        t_g[k] = sp.g[k];
        t_e[k] = sp.energy_K[k];
    }
    for (int k = tid; k < sp.ntrans; k += LOC_SOLVE_THREADS) {
        t_A[k] = sp.A[k];
        t_gr[k] = sp.g[sp.upper[k]] / sp.g[sp.lower[k]];
        t_bg[k] = sp.bgocc[k];
        t_up[k] = sp.upper[k];
        t_lo[k] = sp.lower[k];
    }
    for (int k = tid; k < sp.ncoll; k += LOC_SOLVE_THREADS) {
        t_cu[k] = sp.cu[k];
        t_cl[k] = sp.cl[k];
    }
    for (int k = tid; k < sp.ntemp; k += LOC_SOLVE_THREADS) t_temps[k] = sp.temps[k];
    for (int k = tid; k < sp.ntemp * sp.ncoll; k += LOC_SOLVE_THREADS) t_rates[k] = sp.rates[k];
    __syncthreads();
#define RM(a) Rs[(a) * LOC_SOLVE_THREADS + tid]
#define VX(a) Rs[(NL * NL + (a)) * LOC_SOLVE_THREADS + tid]  // 2 NL more doubles per thread: Boltzmann factors (then the solution)
#define VI(a) Rs[(NL * NL + NL + (a)) * LOC_SOLVE_THREADS + tid]  //   and their inverses
    int64_t i = blockIdx.x * (int64_t)LOC_SOLVE_THREADS + tid;
    bool act = i < n;
    if (act && child && child[i] >= 0) act = false;  // refined cell: no gas of its own
    float rel = 0.0f;
    if (act) {
#pragma unroll
        for (int k = 0; k < NLM * NLM; k++)
            if (k < NL * NL) RM(k) = 0.0;
        const double dens = density[i], T = tkin[i];
        const double ntot = dens * (double)abundance[i];
        // radiative rates: traced transitions from their counters, the others see the background only (DESIGN R23)
        for (int t = 0; t < sp.ntrans; t++) {
            const int u = t_up[t], l = t_lo[t];
            const double gr = t_gr[t];
            double sj = t_bg[t], esc = 1.0;
            for (int k = 0; k < S.nsel; k++)
                if (S.sel[k] == t) {
                    const float2 c = cnt[i * S.nsp + k];
                    sj = c.x;
                    esc = c.y;
                    if (!ali) {  // plain lambda iteration: see k_solve
                        const float2 ke = coef[i * S.nsp + k];
                        if (ke.x != 0.0f) sj += (1.0 - esc) * ((double)ke.y / (double)ke.x);
                        esc = 1.0;
                    }
                }
            const double Aul = t_A[t];
            RM(u * NL + l) += Aul * esc + Aul * sj;  // spontaneous (scaled by the escape probability) + induced
            RM(l * NL + u) += gr * Aul * sj;          // S_lu = B_lu * Jbar
        }
        // collisions: linear interpolation in T, clamped; upward by detailed balance
        int j = 0;
        double f = 0.0;
        if (sp.ntemp > 1) {
            if (T <= t_temps[0]) {
                j = 0;
                f = 0.0;
            } else if (T >= t_temps[sp.ntemp - 1]) {
                j = sp.ntemp - 2;
                f = 1.0;
            } else {
                while (T > t_temps[j + 1]) j++;
                f = (T - t_temps[j]) / (t_temps[j + 1] - t_temps[j]);
            }
        }
        // g_k exp(-(E_k - E_0) / T), once per level
        const double invT = 1.0 / T;
        for (int k = 0; k < NL; k++) {
            const double b = t_g[k] * exp(-(t_e[k] - t_e[0]) * invT);
            VX(k) = b;
            VI(k) = 1.0 / b;  // one division per level instead of one per collisional pair
        }
        for (int k = 0; k < sp.ncoll; k++) {
            const int u = t_cu[k], l = t_cl[k];
            double gd = t_rates[j * sp.ncoll + k];
            if (sp.ntemp > 1) gd = (1.0 - f) * gd + f * t_rates[(j + 1) * sp.ncoll + k];
            RM(u * NL + l) += dens * gd;
            RM(l * NL + u) += dens * (gd * VX(u) * VI(l));
        }
        // GTH elimination
#pragma unroll
        for (int q = NLM - 1; q >= 1; q--) {
            if (q < NL) {
                double sm = 0.0;
#pragma unroll
                for (int c = 0; c < q; c++) sm += RM(q * NL + c);
                const double inv = sm > 0.0 ? 1.0 / sm : 0.0;
#pragma unroll
                for (int r = 0; r < q; r++) {
                    const double rq = RM(r * NL + q) * inv;
                    RM(r * NL + q) = rq;
#pragma unroll
                    for (int c = 0; c < q; c++)
                        if (c != r) RM(r * NL + c) += rq * RM(q * NL + c);
                }
            }
        }
        double x[NLM];
        x[0] = 1.0;
        double tot = 1.0;
#pragma unroll
        for (int q = 1; q < NLM; q++) {
            if (q < NL) {
                double sm = 0.0;
#pragma unroll
                for (int r = 0; r < q; r++) sm += x[r] * RM(r * NL + q);
                x[q] = sm;
                tot += sm;
            }
        }
        const double sc = ntot / tot;
#pragma unroll
        for (int l = 0; l < NLM; l++) {
            if (l < NL) {
                const double nw = x[l] * sc;
                const double old = pops[(int64_t)l * n + i];
                if (ntot > 0.0 && (nw >= 1e-10 * ntot || old >= 1e-10 * ntot))
                    rel = fmaxf(rel, (float)(fabs(nw - old) / fmax(nw, 1e-300)));
                if (!isfinite(nw)) rel = INFINITY;  // see k_solve
                VX(l) = nw;
                pops[(int64_t)l * n + i] = (float)nw;
            }
        }
        // refresh the line coefficients of the traced transitions from the unrounded solution
        for (int k = 0; k < S.nsp; k++) {
            float2 v = make_float2(0.f, 0.f);
            if (k < S.nsel) {
                const double xu = VX(S.upper[k]), xl = VX(S.lower[k]);
                v.x = (float)(S.ck[k] * (xl * (double)S.gratio[k] - xu));
                v.y = (float)(S.ck[k] * xu);
            }
            coef[i * S.nsp + k] = v;
        }
    }
#undef RM
#undef VX
#undef VI
    for (int o = 16; o >= 1; o >>= 1) rel = fmaxf(rel, __shfl_xor_sync(0xffffffffu, rel, o));
    if ((threadIdx.x & 31) == 0 && rel > 0.0f) atomicMax(maxrel_bits, __float_as_uint(rel));
}

// ------------------------------------------------------------------------------------------------
// k_solve_f: the same equations in float32, the rate matrix in REGISTERS (profiles/r2_solve.md).
// One thread per cell, the level count a compile-time constant, every loop unrolled, so that R[u][l] are registers with
// static indices (90 of them at 10 levels; the float64 matrix of k_solve_s needed 960 B of shared memory per cell, which
// left 7 warps per SM and the kernel latency bound at 18 % issue utilisation).  What makes float32 sufficient: the GTH
// elimination has no subtraction, so every population keeps a relative error of ~NL eps = 1e-6 however small it is
// (tolerance of the path: 1e-3); the counters it starts from are float32 sums, and the populations are stored in float32.
// The species enters as DENSE PAIR TABLES in the kernel's parameter space (constant bank: operands of the FMAs, no
// loads): pair p = u (u - 1) / 2 + l for u > l holds the Einstein A of the radiative transition u -> l (0 = none), its
// counter slot (-1 = not ray traced: background only, DESIGN R23), g_u / g_l, the downward collision rate, and
// (E_u - E_l) log2 e: the upward collision rate is gd (g_u/g_l) 2^(-dE2 / T) per PAIR (one ex2 each; the per-level
// Boltzmann factors of the float64 kernels would leave the float32 range for E / T > 87).
// Two things need an index that is only known at run time -- the counter slot of a pair, the levels of a traced
// transition -- and a register array cannot be indexed dynamically: the thread parks its counter record, and later its
// solution, in a column of shared memory (word j of thread t at j * 128 + t: conflict free) and reads it back with the
// run-time index.  Species the tables cannot express (a transition or collisional pair whose upper level has the lower
// index, two radiative transitions between the same levels, more than LOC_SOLVE_F_MAXNL levels) take k_solve_s.
// ------------------------------------------------------------------------------------------------
#define LOC_SOLVE_F_MAXNL 12
#define LOC_SOLVE_F_NPAIR (LOC_SOLVE_F_MAXNL * (LOC_SOLVE_F_MAXNL - 1) / 2)
#define LOC_SOLVE_F_THREADS 128
struct SolveF {
    float A[LOC_SOLVE_F_NPAIR];    // Einstein A of u -> l, 0 = no radiative transition between the pair
    float gr[LOC_SOLVE_F_NPAIR];   // g_u / g_l
    float bg[LOC_SOLVE_F_NPAIR];   // background occupation number at the line frequency
    float dE2[LOC_SOLVE_F_NPAIR];  // (E_u - E_l) log2(e), K
    float gd[LOC_SOLVE_F_NPAIR];   // downward collision rate (ntemp = 1), cm^3/s
    int slot[LOC_SOLVE_F_NPAIR];   // counter slot of the pair's transition, -1 = not traced
    int ntemp, rows;               // rows = scratch words per thread = max(2 nsp, NL)
    float temps[64];
    const float *rates;            // device [ntemp][NL (NL - 1) / 2] dense downward rates (ntemp > 1)
    int nsel, nsp;
    int up[LOC_MAX_TRANS], lo[LOC_MAX_TRANS];
    float ck[LOC_MAX_TRANS], gratio[LOC_MAX_TRANS];
};

// NTI: the collision rates are interpolated in T (ntemp > 1)
template <int NL, bool NTI>
__global__ void __launch_bounds__(LOC_SOLVE_F_THREADS) k_solve_f(int64_t n, const __grid_constant__ SolveF Q, const float *density,
                                                                 const float *tkin, const float *abundance, const float2 *cnt, float *pops,
                                                                 float2 *coef, unsigned int *maxrel_bits, const int32_t *child, int ali)
{
    constexpr int NP = NL * (NL - 1) / 2;
    constexpr int TH = LOC_SOLVE_F_THREADS;
    extern __shared__ __align__(16) float s_f[];
    const int tid = threadIdx.x;
    float *col = s_f + tid;
    const float *s_rates = s_f + Q.rows * TH;
    if (NTI) {
        float *w = s_f + Q.rows * TH;
        for (int k = tid; k < Q.ntemp * NP; k += TH) w[k] = Q.rates[k];
        __syncthreads();
    }
    const int64_t i = blockIdx.x * (int64_t)TH + tid;
    const bool inr = i < n;
    // every global load of the cell is issued here, before anything depends on one (profiles/r2_solve.md: with the loads
    // behind the leaf test and the old populations read at the end, 7.5 issue slots per instruction waited on the long
    // scoreboard): leaf flag, counter record, density / temperature / abundance, old populations
    const int64_t ic = inr ? i : 0;
    const int32_t chd = child ? __ldg(child + ic) : -1;
    const float4 *rec = reinterpret_cast<const float4 *>(cnt + ic * Q.nsp);
    float4 recv[LOC_MAX_TRANS / 2];
#pragma unroll
    for (int h = 0; h < LOC_MAX_TRANS / 2; h++)
        if (2 * h < Q.nsp) recv[h] = __ldg(rec + h);  // (SJ, ESC) of slots 2h, 2h + 1
    const float dens = __ldg(density + ic), T = __ldg(tkin + ic), abun = __ldg(abundance + ic);
    float oldp[NL];
#pragma unroll
    for (int l = 0; l < NL; l++) oldp[l] = pops[(int64_t)l * n + ic];
    const bool act = inr && chd < 0;  // refined cell: no gas of its own
    float rel = 0.0f;
    if (act) {
        // ---- the cell's counter record -> its scratch column ----
        const float4 *crec = reinterpret_cast<const float4 *>(coef + i * Q.nsp);
#pragma unroll
        for (int h = 0; h < LOC_MAX_TRANS / 2; h++) {
            if (2 * h < Q.nsp) {
                float4 v = recv[h];
                if (!ali) {  // plain lambda iteration: see k_solve
                    const float4 ke = crec[h];
                    if (ke.x != 0.0f) v.x += (1.0f - v.y) * (ke.y / ke.x);
                    if (ke.z != 0.0f) v.z += (1.0f - v.w) * (ke.w / ke.z);
                    v.y = 1.0f;
                    v.w = 1.0f;
                }
                col[(4 * h) * TH] = v.x;
                col[(4 * h + 1) * TH] = v.y;
                col[(4 * h + 2) * TH] = v.z;
                col[(4 * h + 3) * TH] = v.w;
            }
        }
        const float ntot = dens * abun;
        // collisions: linear interpolation in T, clamped
        int j = 0;
        float f = 0.0f;
        if (NTI) {
            if (T <= Q.temps[0]) {
                j = 0;
                f = 0.0f;
            } else if (T >= Q.temps[Q.ntemp - 1]) {
                j = Q.ntemp - 2;
                f = 1.0f;
            } else {
                while (T > Q.temps[j + 1]) j++;
                f = (T - Q.temps[j]) / (Q.temps[j + 1] - Q.temps[j]);
            }
        }
        const float nit = -1.0f / T;
        float R[NL][NL];
#pragma unroll
        for (int u = 1; u < NL; u++) {
#pragma unroll
            for (int l = 0; l < u; l++) {
                const int p = u * (u - 1) / 2 + l;
                float gd = Q.gd[p];
                if (NTI) gd = (1.0f - f) * s_rates[j * NP + p] + f * s_rates[(j + 1) * NP + p];
                float dn = dens * gd;
                float upw = dn * Q.gr[p] * ex2f(Q.dE2[p] * nit);  // detailed balance
                if (Q.A[p] != 0.0f) {  // uniform over the grid
                    const int s = Q.slot[p];
                    float sj = Q.bg[p], esc = 1.0f;  // DESIGN R23: untraced transitions see the background only
                    if (s >= 0) {
                        sj = col[(2 * s) * TH];
                        esc = col[(2 * s + 1) * TH];
                    }
                    const float a = Q.A[p];
                    dn += a * esc + a * sj;   // spontaneous (scaled by the escape probability) + induced
                    upw += Q.gr[p] * a * sj;  // S_lu = B_lu * Jbar
                }
                R[u][l] = dn;
                R[l][u] = upw;
            }
        }
        // ---- GTH elimination ----
#pragma unroll
        for (int q = NL - 1; q >= 1; q--) {
            float sm = 0.0f;
#pragma unroll
            for (int c = 0; c < q; c++) sm += R[q][c];
            const float inv = sm > 0.0f ? 1.0f / sm : 0.0f;
#pragma unroll
            for (int r = 0; r < q; r++) {
                const float rq = R[r][q] * inv;
                R[r][q] = rq;
#pragma unroll
                for (int c = 0; c < q; c++)
                    if (c != r) R[r][c] = fmaf(rq, R[q][c], R[r][c]);
            }
        }
        float x[NL];
        x[0] = 1.0f;
        float tot = 1.0f;
#pragma unroll
        for (int q = 1; q < NL; q++) {
            float sm = 0.0f;
#pragma unroll
            for (int r = 0; r < q; r++) sm = fmaf(x[r], R[r][q], sm);
            x[q] = sm;
            tot += sm;
        }
        const float sc = ntot / tot;
#pragma unroll
        for (int l = 0; l < NL; l++) {
            const float nw = x[l] * sc;
            const float old = oldp[l];
            if (ntot > 0.0f && (nw >= 1e-10f * ntot || old >= 1e-10f * ntot)) rel = fmaxf(rel, fabsf(nw - old) / fmaxf(nw, 1e-37f));
            if (!isfinite(nw)) rel = INFINITY;  // see k_solve
            pops[(int64_t)l * n + i] = nw;
            col[l * TH] = nw;
        }
        // ---- line coefficients of the traced transitions for the next iteration ----
        float4 *orec = reinterpret_cast<float4 *>(coef + i * Q.nsp);
#pragma unroll
        for (int h = 0; h < LOC_MAX_TRANS / 2; h++) {
            if (2 * h < Q.nsp) {
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (2 * h < Q.nsel) {
                    const float xu = col[Q.up[2 * h] * TH], xl = col[Q.lo[2 * h] * TH];
                    v.x = Q.ck[2 * h] * (xl * Q.gratio[2 * h] - xu);
                    v.y = Q.ck[2 * h] * xu;
                }
                if (2 * h + 1 < Q.nsel) {
                    const float xu = col[Q.up[2 * h + 1] * TH], xl = col[Q.lo[2 * h + 1] * TH];
                    v.z = Q.ck[2 * h + 1] * (xl * Q.gratio[2 * h + 1] - xu);
                    v.w = Q.ck[2 * h + 1] * xu;
                }
                orec[h] = v;
            }
        }
    }
    for (int o = 16; o >= 1; o >>= 1) rel = fmaxf(rel, __shfl_xor_sync(0xffffffffu, rel, o));
    if ((threadIdx.x & 31) == 0 && rel > 0.0f) atomicMax(maxrel_bits, __float_as_uint(rel));
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
// dense pair tables of k_solve_f from the species and the current selection.  Returns 1 = filled, 0 = the species does not
// fit them (the float64 kernels take over), LOC_ECUDA = the upload of the dense rate table failed (reported, never hidden
// behind the fallback).
static int fill_solve_f(loc_model *m, SolveF &Q)
{
    const int NL = m->nlevel;
    if (NL < 2 || NL > LOC_SOLVE_F_MAXNL) return 0;
    memset(&Q, 0, sizeof(Q));
    const int np = NL * (NL - 1) / 2;
    for (int u = 1; u < NL; u++)
        for (int l = 0; l < u; l++) {
            const int p = u * (u - 1) / 2 + l;
            Q.gr[p] = (float)(m->h_g[u] / m->h_g[l]);
            Q.dE2[p] = (float)((m->h_energy[u] - m->h_energy[l]) * 1.4426950408889634);
            Q.slot[p] = -1;
        }
    for (int t = 0; t < m->ntrans; t++) {
        const int u = m->h_upper[t], l = m->h_lower[t];
        if (u <= l) return 0;
        const int p = u * (u - 1) / 2 + l;
        if (Q.A[p] != 0.0f) return 0;  // two transitions between the same levels
        Q.A[p] = (float)m->h_A[t];
        if (Q.A[p] == 0.0f) return 0;  // below the float32 range
        Q.bg[p] = (m->tbg > 0.0) ? (float)(1.0 / expm1(LOC_HP * m->h_freq[t] / (LOC_KB * m->tbg))) : 0.0f;
        for (int k = 0; k < m->selh.nsel; k++)
            if (m->selh.sel[k] == t) Q.slot[p] = k;
    }
    std::vector<float> dense((size_t)m->ntemp * np, 0.0f);
    for (int k = 0; k < m->ncoll; k++) {
        const int u = m->h_cu[k], l = m->h_cl[k];
        if (u <= l) return 0;
        const int p = u * (u - 1) / 2 + l;
        for (int j = 0; j < m->ntemp; j++) dense[(size_t)j * np + p] += (float)m->h_rates[(size_t)j * m->ncoll + k];
    }
    Q.ntemp = m->ntemp;
    if (m->ntemp == 1) {
        for (int p = 0; p < np; p++) Q.gd[p] = dense[p];
    } else {
        for (int j = 0; j < m->ntemp; j++) Q.temps[j] = (float)m->h_temps[j];
        // the dense table lives in the workspace; rewritten only when the species changes (loc_set_species clears the flag).
        // The first solve after loc_set_species therefore waits once for the stream (`dense` goes out of scope).
        if (!m->rates_f_valid) {
            LOC_CUDA_CHECK(m, cudaMemcpyAsync(m->d_rates_f, dense.data(), sizeof(float) * dense.size(), cudaMemcpyHostToDevice, m->stream));
            LOC_CUDA_CHECK(m, cudaStreamSynchronize(m->stream));
            m->rates_f_valid = true;
        }
        Q.rates = m->d_rates_f;
    }
    Q.nsel = m->selh.nsel;
    Q.nsp = m->selh.nsp;
    Q.rows = std::max(2 * Q.nsp, NL);
    for (int k = 0; k < Q.nsel; k++) {
        Q.up[k] = m->selh.upper[k];
        Q.lo[k] = m->selh.lower[k];
        Q.ck[k] = (float)m->selh.ck[k];
        Q.gratio[k] = m->selh.gratio[k];
    }
    return 1;
}

template <int NL>
static int launch_solve_f(loc_model *m, const SolveF &Q, const int32_t *ch)
{
    const int64_t n = m->ncell;
    const size_t smem = sizeof(float) * ((size_t)Q.rows * LOC_SOLVE_F_THREADS + (Q.ntemp > 1 ? (size_t)Q.ntemp * NL * (NL - 1) / 2 : 0));
    const unsigned nb = (unsigned)((n + LOC_SOLVE_F_THREADS - 1) / LOC_SOLVE_F_THREADS);
    if (Q.ntemp > 1) {
        LOC_CUDA_CHECK(m, cudaFuncSetAttribute(k_solve_f<NL, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        k_solve_f<NL, true><<<nb, LOC_SOLVE_F_THREADS, smem, m->stream>>>(n, Q, m->cells.density, m->cells.tkin, m->cells.abundance, m->cnt,
                                                                         m->pops, m->coef, m->d_maxrel, ch, m->ali);
    } else {
        k_solve_f<NL, false><<<nb, LOC_SOLVE_F_THREADS, smem, m->stream>>>(n, Q, m->cells.density, m->cells.tkin, m->cells.abundance, m->cnt,
                                                                          m->pops, m->coef, m->d_maxrel, ch, m->ali);
    }
    return LOC_OK;
}

// S8 over all cells from the current counters; refreshes the line coefficients.  Asynchronous.
int loc_launch_solve(loc_model *m)
{
    int64_t n = m->ncell;
    const int32_t *ch = m->kind == LOC_GRID_OCTREE ? m->child : nullptr;
    // loc_set_option(LOC_OPT_SOLVER): 0 = automatic (float32 registers where the species fits, else float64 in shared
    // memory, else float64 in local memory), 1 = force the local-memory kernel, 2 = the shared-memory kernel (A/B runs)
    if (m->solver == 0) {
        SolveF Q;
        const int fits = fill_solve_f(m, Q);
        if (fits < 0) return fits;
        if (fits) {
            int rc = LOC_EINVAL;
            switch (m->nlevel) {
#define LOC_SF(N)                          \
    case N:                                \
        rc = launch_solve_f<N>(m, Q, ch);  \
        break;
                LOC_SF(2) LOC_SF(3) LOC_SF(4) LOC_SF(5) LOC_SF(6) LOC_SF(7) LOC_SF(8) LOC_SF(9) LOC_SF(10) LOC_SF(11) LOC_SF(12)
#undef LOC_SF
            }
            if (rc != LOC_OK) return rc;
            m->launches++;
            LOC_CUDA_CHECK(m, cudaGetLastError());
            m->coef_valid = true;
            return LOC_OK;
        }
    }
    unsigned nb = (unsigned)((n + 127) / 128);
#define LOC_SOLVE(NLMAX)                                                                                                     \
    k_solve<NLMAX><<<nb, 128, 0, m->stream>>>(n, m->sp, m->selh, m->cells.density, m->cells.tkin, m->cells.abundance, m->cnt, \
                                              m->pops, m->coef, m->d_maxrel, ch, m->ali)
    // float64: the shared-memory kernel while a block's matrices and the species tables fit, else the local-memory kernel
    {
        const int NL = m->nlevel;
        SolveTabs T;
        int o = 0;
        auto take = [&](int bytes) {
            int at = o;
            o += (bytes + 7) & ~7;
            return at;
        };
        T.g = take(8 * NL);
        T.energy = take(8 * NL);
        T.A = take(8 * m->ntrans);
        T.bg = take(8 * m->ntrans);
        T.gr = take(8 * m->ntrans);
        T.temps = take(8 * m->ntemp);
        T.rates = take(8 * m->ntemp * m->ncoll);
        T.upper = take(4 * m->ntrans);
        T.lower = take(4 * m->ntrans);
        T.cu = take(4 * m->ncoll);
        T.cl = take(4 * m->ncoll);
        T.bytes = o;
        const size_t smem = sizeof(double) * (size_t)(NL * NL + 2 * NL) * LOC_SOLVE_THREADS + (size_t)o;
        if (NL <= 16 && smem <= 200 * 1024 && m->solver != 1) {
            const unsigned nbs = (unsigned)((n + LOC_SOLVE_THREADS - 1) / LOC_SOLVE_THREADS);
#define LOC_SOLVE_S(NLX)                                                                                                          \
    do {                                                                                                                          \
        LOC_CUDA_CHECK(m, cudaFuncSetAttribute(k_solve_s<NLX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));          \
        k_solve_s<NLX><<<nbs, LOC_SOLVE_THREADS, smem, m->stream>>>(n, m->sp, m->selh, m->cells.density, m->cells.tkin,          \
                                                                    m->cells.abundance, m->cnt, m->pops, m->coef, m->d_maxrel, ch, \
                                                                    m->ali, T);                                                   \
    } while (0)
            if (NL == 10) LOC_SOLVE_S(10);
            else if (NL == 5) LOC_SOLVE_S(5);
            else if (NL == 4) LOC_SOLVE_S(4);
            else LOC_SOLVE_S(0);
#undef LOC_SOLVE_S
            m->launches++;
            LOC_CUDA_CHECK(m, cudaGetLastError());
            m->coef_valid = true;
            return LOC_OK;
        }
    }
    if (m->nlevel <= 6) LOC_SOLVE(6);
    else if (m->nlevel <= 10) LOC_SOLVE(10);
    else if (m->nlevel <= 16) LOC_SOLVE(16);
    else LOC_SOLVE(32);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    m->coef_valid = true;
    return LOC_OK;
}
