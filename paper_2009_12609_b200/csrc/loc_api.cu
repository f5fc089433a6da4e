// loc_api.cu -- C-ABI entry points (include/loc.h), host-side set-up, and the small per-cell kernels:
// kinematics packing, LTE initialisation, line coefficients, statistical-equilibrium solve.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "loc_internal.cuh"

static char g_create_err[512] = "";

// ------------------------------------------------------------------------------------------------
// workspace carving
// ------------------------------------------------------------------------------------------------
static inline int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

struct Carver {
    char *base;
    int64_t off, cap;
    bool dry;
    template <typename T>
    T *take(int64_t n)
    {
        off = align_up(off, 256);
        T *p = dry ? nullptr : reinterpret_cast<T *>(base + off);
        off += n * (int64_t)sizeof(T);
        return p;
    }
};

// multiprocessors of the current device; 148 (B200) only when no device can be queried (sizing calls without a GPU)
static int device_sm_count()
{
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1) {
        cudaGetLastError();
        return 148;
    }
    return nsm;
}
static int max_resident_ctas() { return device_sm_count() * 16; }  // upper bound used to size the per-CTA spectrum slots

// lays out the workspace; with dry=true only sizes are computed
static int64_t carve(loc_model *m, Carver &c, const loc_grid *g, int nch, int nlevel, int ntrans, int ndir_max)
{
    int64_t ncell = (g->kind == LOC_GRID_SHELL) ? g->nshell : g->level_offset[g->nlevel];
    int nsp = (ntrans + 1) & ~1;
    m->kin = c.take<float4>(ncell);
    m->coef = c.take<float2>(ncell * nsp);
    m->cnt = c.take<float2>(ncell * nsp);
    m->visits = c.take<uint32_t>(ncell);
    m->pathz = c.take<uint32_t>(ncell);
    m->d_steps = c.take<unsigned long long>(4);  // [0] steps, [1] active channels (5 sigma rule), [2..3] scratch
    m->d_maxrel = c.take<unsigned int>(1);
    m->d_errflag = c.take<int>(1);
    m->d_queue = c.take<unsigned int>(1);
    // species arrays
    int ncoll = nlevel * (nlevel - 1) / 2;
    int ntall = std::max(ntrans, ncoll);  // the species may hold more radiative transitions than are traced
    m->sp.energy_K = c.take<double>(nlevel);
    m->sp.g = c.take<double>(nlevel);
    m->sp.upper = c.take<int>(ntall);
    m->sp.lower = c.take<int>(ntall);
    m->sp.A = c.take<double>(ntall);
    m->sp.freq = c.take<double>(ntall);
    m->sp.bgocc = c.take<double>(ntall);
    m->sp.cu = c.take<int>(ncoll);
    m->sp.cl = c.take<int>(ncoll);
    m->sp.temps = c.take<double>(64);
    m->sp.rates = c.take<double>((int64_t)64 * ncoll);
    if (g->kind == LOC_GRID_SHELL) {
        int64_t ntab = 0;
        // triangular tables: ray i with tangent shell k0 has nshell-k0 entries; bound by nray*nshell
        ntab = (int64_t)g->nray * g->nshell;
        m->d_order = c.take<int>(g->nray);
        m->d_k0 = c.take<int>(g->nray);
        m->d_off = c.take<long long>(g->nray);
        m->d_tabs = c.take<float>(ntab);
        m->d_tabmu = c.take<float>(ntab);
        m->d_tabw = c.take<float>(ntab);
        m->d_rout = c.take<double>(g->nshell);
    } else {
        // root-line tasks: at most max(face) lines per direction
        int64_t face = std::max((int64_t)g->nx * g->ny, std::max((int64_t)g->ny * g->nz, (int64_t)g->nx * g->nz));
        m->ntask_max = face * ndir_max;
        m->d_dirs = c.take<Dir3>(ndir_max);
        m->d_task_off = c.take<long long>(m->ntask_max + 1);
        m->d_task_dir = c.take<uint16_t>(m->ntask_max);
        // step stream: every leaf is crossed by (1 + s_p + s_q) <= 3 ray segments per direction on average;
        // control records (background / save / load) ride in the same bound
        m->stream_cap = 3 * ncell * (int64_t)ndir_max + 16 * m->ntask_max + 1024;
        m->d_stream = c.take<uint2>(m->stream_cap);
        m->bstack_threads = (int)std::min<int64_t>(m->ntask_max, LOC_BUILD_BATCH);
        m->d_bstack = c.take<char>((int64_t)m->bstack_threads * LOC_BUILD_STACK * 16);
        m->max_warps = max_resident_ctas();
        m->spec_pool_floats = (int64_t)m->max_warps * 4 * std::max(g->nlevel - 1, 1) * nsp * ((nch + 3) & ~3);  // 4 rays per warp
        m->spec_pool = c.take<float>(m->spec_pool_floats);
    }
    return align_up(c.off, 256);
}

extern "C" int64_t loc_workspace_bytes(const loc_grid *g, int nchannel, int nlevel_species, int ntrans, int ndir_max)
{
    if (!g || nchannel < 1 || nlevel_species < 2 || nlevel_species > LOC_MAX_LEVELS || ntrans < 1 || ndir_max > LOC_MAX_DIRS) return LOC_EINVAL;
    if (g->kind == LOC_GRID_SHELL) {
        if (g->nshell < 1 || g->nray < 1) return LOC_EINVAL;
    } else if (g->kind == LOC_GRID_OCTREE) {
        if (g->nlevel < 1 || g->nlevel > LOC_MAXL || !g->level_offset) return LOC_EINVAL;
    } else
        return LOC_EINVAL;
    loc_model tmp;
    memset(&tmp, 0, sizeof(tmp));
    Carver c{nullptr, 0, 0, true};
    return carve(&tmp, c, g, nchannel, nlevel_species, std::min(ntrans, LOC_MAX_TRANS), std::max(ndir_max, 1));
}

// ------------------------------------------------------------------------------------------------
// small kernels
// ------------------------------------------------------------------------------------------------
__global__ void k_pack_kin(int64_t n, const float *vx, const float *vy, const float *vz, const float *sigma, const float *tkin,
                           double kT_over_m_per_K, float4 *kin)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double s = sigma[i];
    double st = sqrt(s * s + kT_over_m_per_K * (double)tkin[i]);  // DESIGN R3
    kin[i] = make_float4(vx[i], vy ? vy[i] : 0.0f, vz ? vz[i] : 0.0f, (float)st);
}

__global__ void k_lte(int64_t n, SpeciesDev sp, const float *density, const float *tkin, const float *abundance, float *pops)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double T = tkin[i], Z = 0.0;
    for (int l = 0; l < sp.nlevel; l++) Z += sp.g[l] * exp(-sp.energy_K[l] / T);
    double ntot = (double)density[i] * (double)abundance[i];
    for (int l = 0; l < sp.nlevel; l++) pops[(int64_t)l * n + i] = (float)(ntot * sp.g[l] * exp(-sp.energy_K[l] / T) / Z);
}

// line coefficients of the traced transitions from the populations (DESIGN 5.2):
//   kap = C_t (n_l g_u/g_l - n_u)   [1/cm per unit profile fraction],   em = C_t n_u,   C_t = c^3 A/(8 pi nu^3 dv)
__global__ void k_coef(int64_t n, Selection S, const float *pops, float2 *coef)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    for (int k = 0; k < S.nsp; k++) {
        float2 v = make_float2(0.f, 0.f);
        if (k < S.nsel) {
            double nu_ = pops[(int64_t)S.upper[k] * n + i], nl_ = pops[(int64_t)S.lower[k] * n + i];
            v.x = (float)(S.ck[k] * (nl_ * (double)S.gratio[k] - nu_));
            v.y = (float)(S.ck[k] * nu_);
        }
        coef[i * S.nsp + k] = v;
    }
}

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
// helpers
// ------------------------------------------------------------------------------------------------
static int fail(loc_model *m, int code, const char *msg)
{
    snprintf(m ? m->err : g_create_err, 512, "%s", msg);
    return code;
}

static int build_selection(loc_model *m, int nsel, const int *idx)
{
    Selection &S = m->selh;
    if (nsel == 0) {
        // default selection: the first transitions, as many as the model was created for (the per-cell records of the
        // workspace hold max_trans entries)
        nsel = std::min(std::min(m->ntrans, LOC_MAX_TRANS), m->max_trans);
        for (int k = 0; k < nsel; k++) S.sel[k] = k;
    } else {
        if (nsel < 0 || nsel > LOC_MAX_TRANS || nsel > m->max_trans) return fail(m, LOC_EINVAL, "loc_simulate: nsel out of range");
        for (int k = 0; k < nsel; k++) {
            if (idx[k] < 0 || idx[k] >= m->ntrans) return fail(m, LOC_EINVAL, "loc_simulate: transition index out of range");
            S.sel[k] = idx[k];
        }
    }
    bool changed = (S.nsel != nsel);
    S.nsel = nsel;
    S.nsp = (nsel + 1) & ~1;
    for (int k = 0; k < nsel; k++) {
        int t = S.sel[k];
        int u = m->h_upper[t], l = m->h_lower[t];
        if (S.upper[k] != u || S.lower[k] != l) changed = true;
        S.upper[k] = u;
        S.lower[k] = l;
        S.gratio[k] = (float)(m->h_g[u] / m->h_g[l]);
        double nu = m->h_freq[t];
        S.ck[k] = LOC_CL * LOC_CL * LOC_CL * m->h_A[t] / (8.0 * LOC_PI * nu * nu * nu * m->dv);
        S.bgocc[k] = (m->tbg > 0.0) ? (float)(1.0 / expm1(LOC_HP * nu / (LOC_KB * m->tbg))) : 0.0f;
    }
    if (changed) m->coef_valid = false;
    return LOC_OK;
}

static int refresh_coef(loc_model *m)
{
    if (!m->pops) return fail(m, LOC_ESTATE, "populations not registered (loc_set_populations / loc_init_lte)");
    int64_t n = m->ncell;
    k_coef<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(n, m->selh, m->pops, m->coef);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    m->coef_valid = true;
    return LOC_OK;
}

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
extern "C" int loc_create_model(const loc_grid *g, const loc_cells *cells, int nchannel, double band_half, double tbg,
                                int nlevel_max, int ntrans_max, int ndir_max, void *workspace, int64_t workspace_bytes, void *stream, loc_model **out)
{
    if (!out) return fail(nullptr, LOC_EINVAL, "out is NULL");
    *out = nullptr;
    if (!g || !cells || !workspace) return fail(nullptr, LOC_EINVAL, "NULL argument");
    if (nchannel < 1 || nchannel > 1024) return fail(nullptr, LOC_EINVAL, "nchannel must be in [1,1024]");
    if (nlevel_max < 2 || nlevel_max > LOC_MAX_LEVELS || ntrans_max < 1) return fail(nullptr, LOC_EINVAL, "species limits out of range");
    if (ndir_max > LOC_MAX_DIRS) return fail(nullptr, LOC_EINVAL, "ndir_max exceeds 65535 directions");
    if (!(band_half > 0.0) || tbg < 0.0) return fail(nullptr, LOC_EINVAL, "band_halfwidth must be > 0 and t_background >= 0");
    if (!cells->density || !cells->tkin || !cells->sigma || !cells->vx || !cells->abundance)
        return fail(nullptr, LOC_EINVAL, "cell arrays missing");
    if (g->kind == LOC_GRID_SHELL) {
        if (g->nshell < 1 || g->nray < 1 || !g->r_out || !g->ray_p || !g->ray_w) return fail(nullptr, LOC_EINVAL, "shell grid incomplete");
        double prev = 0.0;
        for (int k = 0; k < g->nshell; k++) {
            if (!(g->r_out[k] > prev)) return fail(nullptr, LOC_EINVAL, "shell radii must be positive and strictly ascending");
            prev = g->r_out[k];
        }
        for (int i = 0; i < g->nray; i++)
            if (!(g->ray_p[i] >= 0.0) || !(g->ray_p[i] < g->r_out[g->nshell - 1]) || !(g->ray_w[i] > 0.0))
                return fail(nullptr, LOC_EINVAL, "ray impact parameter outside the model or weight <= 0");
    } else if (g->kind == LOC_GRID_OCTREE) {
        if (g->nx < 1 || g->ny < 1 || g->nz < 1 || g->nx > 1024 || g->ny > 1024 || g->nz > 1024 || !(g->root_cell_cm > 0.0))
            return fail(nullptr, LOC_EINVAL, "root grid dimensions must be in [1,1024] and root_cell_cm > 0");
        if (g->nlevel < 1 || g->nlevel > LOC_MAXL || !g->level_offset || !g->child) return fail(nullptr, LOC_EINVAL, "octree hierarchy incomplete");
        if (g->level_offset[0] != 0 || g->level_offset[1] != (int64_t)g->nx * g->ny * g->nz)
            return fail(nullptr, LOC_EINVAL, "level_offset[1] must equal nx*ny*nz");
        for (int l = 1; l < g->nlevel; l++)
            if ((g->level_offset[l + 1] - g->level_offset[l]) % 8 != 0 || g->level_offset[l + 1] < g->level_offset[l])
                return fail(nullptr, LOC_EINVAL, "refined levels must hold whole octets");
        if (g->level_offset[g->nlevel] >= ((int64_t)1 << 31)) return fail(nullptr, LOC_EINVAL, "more than 2^31 cells");
    } else
        return fail(nullptr, LOC_EINVAL, "unknown grid kind");

    loc_model *m = new (std::nothrow) loc_model;
    if (!m) return fail(nullptr, LOC_ENOMEM, "host allocation failed");
    memset(m, 0, sizeof(*m));
    m->kind = g->kind;
    m->stream = (cudaStream_t)stream;
    m->nch = nchannel;
    m->band_half = band_half;
    m->dv = 2.0 * band_half / nchannel;
    m->tbg = tbg;
    m->cells = *cells;
    m->xmin = 4.5f;
    m->ali = 1;
    m->eps_tau = 1e-6f;
    m->xclip = LOC_XCLIP;
    m->nsm = device_sm_count();
    m->ncell = (g->kind == LOC_GRID_SHELL) ? g->nshell : g->level_offset[g->nlevel];
    m->ws = (char *)workspace;
    m->ws_bytes = workspace_bytes;
    int best_nt = std::min(ntrans_max, LOC_MAX_TRANS), best_nd = std::max(ndir_max, 1);
    {
        loc_model tmp;
        memset(&tmp, 0, sizeof(tmp));
        Carver c{nullptr, 0, 0, true};
        if (carve(&tmp, c, g, nchannel, nlevel_max, best_nt, best_nd) > workspace_bytes) {
            delete m;
            return fail(nullptr, LOC_ENOMEM, "workspace too small (see loc_workspace_bytes)");
        }
    }
    m->max_trans = best_nt;
    m->ndir_max = best_nd;
    Carver c{m->ws, 0, workspace_bytes, false};
    m->ws_used = carve(m, c, g, nchannel, nlevel_max, best_nt, best_nd);
    m->max_levels = nlevel_max;

    cudaError_t e;
    if ((e = cudaMemsetAsync(m->d_errflag, 0, sizeof(int), m->stream)) != cudaSuccess ||
        (e = cudaMemsetAsync(m->d_maxrel, 0, sizeof(unsigned int), m->stream)) != cudaSuccess ||
        (e = cudaMemsetAsync(m->d_steps, 0, 2 * sizeof(unsigned long long), m->stream)) != cudaSuccess) {
        snprintf(g_create_err, 512, "cudaMemsetAsync: %s", cudaGetErrorString(e));
        delete m;
        return LOC_ECUDA;
    }
    if (g->kind == LOC_GRID_SHELL) {
        m->nshell = g->nshell;
        m->nray = g->nray;
        int ns = g->nshell, nr = g->nray;
        m->h_rout = (double *)malloc(sizeof(double) * ns);
        memcpy(m->h_rout, g->r_out, sizeof(double) * ns);
        // S0 set-up tables ("The distance that a ray travels through each shell is pre-calculated")
        std::vector<int> k0(nr), order(nr);
        std::vector<long long> off(nr);
        std::vector<double> veff(ns, 0.0);
        std::vector<float> tabs, tabmu, tabw;
        tabs.reserve((size_t)nr * ns / 2 + nr);
        tabmu.reserve((size_t)nr * ns / 2 + nr);
        int64_t steps = 0;
        for (int i = 0; i < nr; i++) {
            double p = g->ray_p[i];
            int k = 0;
            while (k < ns - 1 && p >= g->r_out[k]) k++;
            k0[i] = k;
            off[i] = (long long)tabs.size();
            for (int kk = k; kk < ns; kk++) {
                double ro = g->r_out[kk], ri = (kk > 0) ? g->r_out[kk - 1] : 0.0;
                double s = (kk == k) ? 2.0 * sqrt(ro * ro - p * p) : sqrt(ro * ro - p * p) - sqrt(ri * ri - p * p);
                double mu = sqrt(1.0 - p * p / (ro * ro));
                tabs.push_back((float)s);
                tabmu.push_back((float)mu);
                veff[kk] += g->ray_w[i] * s * ((kk == k) ? 1.0 : 2.0);  // DESIGN R12: V_eff = sum_i W_i s_ik, both crossings
            }
            steps += 2 * (ns - 1 - k) + 1;
        }
        m->steps1d = steps;
        // this ray's share W_i s_ik / V_eff,k of the shell, formed in double: the factors themselves (~1e34 cm^2,
        // ~1e17 cm, ~1e-52 cm^-3) leave the float32 range
        tabw.resize(tabs.size());
        for (int i = 0; i < nr; i++)
            for (int kk = k0[i]; kk < ns; kk++) {
                double ro = g->r_out[kk], ri = (kk > 0) ? g->r_out[kk - 1] : 0.0, p = g->ray_p[i];
                double sd = (kk == k0[i]) ? 2.0 * sqrt(ro * ro - p * p) : sqrt(ro * ro - p * p) - sqrt(ri * ri - p * p);
                tabw[off[i] + (kk - k0[i])] = veff[kk] > 0.0 ? (float)(g->ray_w[i] * sd / veff[kk]) : 0.0f;
            }
        for (int i = 0; i < nr; i++) order[i] = i;
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return k0[a] < k0[b]; });  // longest rays first
        if ((int64_t)tabs.size() > (int64_t)nr * ns) {
            delete m;
            return fail(nullptr, LOC_ENOMEM, "internal: path table larger than carved");
        }
#define H2D(dst, src, bytes)                                                                           \
    if ((e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, m->stream)) != cudaSuccess) {     \
        snprintf(g_create_err, 512, "cudaMemcpyAsync: %s", cudaGetErrorString(e));                      \
        delete m;                                                                                       \
        return LOC_ECUDA;                                                                               \
    }
        H2D(m->d_order, order.data(), sizeof(int) * nr);
        H2D(m->d_k0, k0.data(), sizeof(int) * nr);
        H2D(m->d_off, off.data(), sizeof(long long) * nr);
        H2D(m->d_tabs, tabs.data(), sizeof(float) * tabs.size());
        H2D(m->d_tabmu, tabmu.data(), sizeof(float) * tabmu.size());
        H2D(m->d_tabw, tabw.data(), sizeof(float) * tabw.size());
        H2D(m->d_rout, g->r_out, sizeof(double) * ns);
        cudaStreamSynchronize(m->stream);  // host vectors go out of scope
    } else {
        m->nx = g->nx;
        m->ny = g->ny;
        m->nz = g->nz;
        m->nlev = g->nlevel;
        m->root_cm = g->root_cell_cm;
        for (int l = 0; l <= g->nlevel; l++) m->noff[l] = g->level_offset[l];
        m->child = g->child;
        m->h_dirs = (Dir3 *)malloc(sizeof(Dir3) * m->ndir_max);
        int rc = loc_setup3d(m);
        if (rc != LOC_OK) {
            snprintf(g_create_err, 512, "%s", m->err);
            loc_destroy_model(m);
            return rc;
        }
    }
    *out = m;
    return LOC_OK;
}

// kinematics record: (vx, vy, vz, total sigma) with the thermal broadening k T / m added (DESIGN R3)
extern "C" int loc_refresh_cells(loc_model *m)
{
    if (!m) return LOC_EINVAL;
    if (!m->have_species) return fail(m, LOC_ESTATE, "loc_set_species must be called first");
    double ktm = (m->sp.mass_amu > 0.0) ? LOC_KB / (m->sp.mass_amu * LOC_AMU) : 0.0;
    int64_t n = m->ncell;
    k_pack_kin<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(n, m->cells.vx, m->kind == LOC_GRID_OCTREE ? m->cells.vy : nullptr,
                                                                  m->kind == LOC_GRID_OCTREE ? m->cells.vz : nullptr, m->cells.sigma,
                                                                  m->cells.tkin, ktm, m->kin);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    return LOC_OK;
}

extern "C" int loc_set_species(loc_model *m, int nlevel, const double *energy_K, const double *g, int ntrans, const int *upper,
                               const int *lower, const double *A, double mass_amu, int ncoll, const int *cu, const int *cl,
                               int ntemp, const double *temps_K, const double *rate_down)
{
    if (!m) return LOC_EINVAL;
    if (nlevel < 2 || nlevel > LOC_MAX_LEVELS || nlevel > m->max_levels) return fail(m, LOC_EINVAL, "nlevel must be in [2,32] and within the limit given to loc_create_model");
    if (ntrans < 1 || ntrans > nlevel * (nlevel - 1) / 2) return fail(m, LOC_EINVAL, "ntrans out of range");
    if (ncoll < 0 || ncoll > nlevel * (nlevel - 1) / 2) return fail(m, LOC_EINVAL, "ncoll out of range");
    if (ntemp < 1 || ntemp > 64) return fail(m, LOC_EINVAL, "ntemp must be in [1,64]");
    if (!energy_K || !g || !upper || !lower || !A || (ncoll && (!cu || !cl || !temps_K || !rate_down))) return fail(m, LOC_EINVAL, "NULL species array");
    for (int t = 0; t < ntrans; t++) {
        if (upper[t] < 0 || upper[t] >= nlevel || lower[t] < 0 || lower[t] >= nlevel || !(energy_K[upper[t]] > energy_K[lower[t]]) || !(A[t] > 0))
            return fail(m, LOC_EINVAL, "bad radiative transition");
    }
    for (int k = 0; k < ncoll; k++)
        if (cu[k] < 0 || cu[k] >= nlevel || cl[k] < 0 || cl[k] >= nlevel || cu[k] == cl[k]) return fail(m, LOC_EINVAL, "bad collisional pair");
    for (int j = 1; j < ntemp; j++)
        if (!(temps_K[j] > temps_K[j - 1])) return fail(m, LOC_EINVAL, "collision temperatures must ascend");
    m->nlevel = nlevel;
    m->ntrans = ntrans;
    m->ncoll = ncoll;
    m->ntemp = ntemp;
    memcpy(m->h_energy, energy_K, sizeof(double) * nlevel);
    memcpy(m->h_g, g, sizeof(double) * nlevel);
    free(m->h_upper); free(m->h_lower); free(m->h_A); free(m->h_freq);
    m->h_upper = (int *)malloc(sizeof(int) * ntrans);
    m->h_lower = (int *)malloc(sizeof(int) * ntrans);
    m->h_A = (double *)malloc(sizeof(double) * ntrans);
    m->h_freq = (double *)malloc(sizeof(double) * ntrans);
    std::vector<double> bg(ntrans);
    for (int t = 0; t < ntrans; t++) {
        m->h_upper[t] = upper[t];
        m->h_lower[t] = lower[t];
        m->h_A[t] = A[t];
        m->h_freq[t] = (energy_K[upper[t]] - energy_K[lower[t]]) * LOC_KB / LOC_HP;
        bg[t] = (m->tbg > 0.0) ? 1.0 / expm1(LOC_HP * m->h_freq[t] / (LOC_KB * m->tbg)) : 0.0;
    }
    SpeciesDev &sp = m->sp;
    sp.nlevel = nlevel;
    sp.ntrans = ntrans;
    sp.ncoll = ncoll;
    sp.ntemp = ntemp;
    sp.mass_amu = mass_amu;
    cudaStream_t st = m->stream;
    LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.energy_K, energy_K, sizeof(double) * nlevel, cudaMemcpyHostToDevice, st));
    LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.g, g, sizeof(double) * nlevel, cudaMemcpyHostToDevice, st));
    LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.upper, upper, sizeof(int) * ntrans, cudaMemcpyHostToDevice, st));
    LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.lower, lower, sizeof(int) * ntrans, cudaMemcpyHostToDevice, st));
    LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.A, A, sizeof(double) * ntrans, cudaMemcpyHostToDevice, st));
    LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.freq, m->h_freq, sizeof(double) * ntrans, cudaMemcpyHostToDevice, st));
    LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.bgocc, bg.data(), sizeof(double) * ntrans, cudaMemcpyHostToDevice, st));
    if (ncoll) {
        LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.cu, cu, sizeof(int) * ncoll, cudaMemcpyHostToDevice, st));
        LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.cl, cl, sizeof(int) * ncoll, cudaMemcpyHostToDevice, st));
        LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.temps, temps_K, sizeof(double) * ntemp, cudaMemcpyHostToDevice, st));
        LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.rates, rate_down, sizeof(double) * ntemp * ncoll, cudaMemcpyHostToDevice, st));
    }
    m->have_species = true;
    {
        int rc = loc_refresh_cells(m);
        if (rc) return rc;
    }
    LOC_CUDA_CHECK(m, cudaStreamSynchronize(st));  // bg vector goes out of scope
    m->have_species = true;
    m->selh.nsel = 0;
    m->coef_valid = false;
    return build_selection(m, 0, nullptr);
}

extern "C" int loc_set_directions(loc_model *m, int ndir, const double *dir)
{
    if (!m || !dir) return LOC_EINVAL;
    if (m->kind != LOC_GRID_OCTREE) return fail(m, LOC_ESTATE, "loc_set_directions: octree models only");
    if (ndir < 1 || ndir > m->ndir_max) return fail(m, LOC_EINVAL, "ndir exceeds the ndir_max the workspace was sized for");
    for (int i = 0; i < ndir; i++) {
        const double *d = dir + 3 * i;
        double nn = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
        if (!(fabs(nn - 1.0) < 1e-9)) return fail(m, LOC_EINVAL, "direction is not a unit vector");
    }
    // the model has NO directions until the new step stream is complete: a failure below (LOC_ENOMEM, LOC_ECUDA) leaves
    // loc_simulate refusing to run (LOC_ESTATE) instead of replaying a half-written stream
    m->ndir = 0;
    m->ntask = 0;
    m->stream_len = 0;
    m->setup_steps = 0;
    m->simulated = false;
    int64_t t0 = 0;
    for (int i = 0; i < ndir; i++) {
        loc_fill_dir(m, dir + 3 * i, &m->h_dirs[i]);
        m->h_dirs[i].task0 = t0;
        t0 += (int64_t)m->h_dirs[i].np * m->h_dirs[i].nq;
    }
    LOC_CUDA_CHECK(m, cudaMemcpyAsync(m->d_dirs, m->h_dirs, sizeof(Dir3) * ndir, cudaMemcpyHostToDevice, m->stream));
    LOC_CUDA_CHECK(m, cudaStreamSynchronize(m->stream));
    const int rc = loc_build_streams(m, ndir, t0);  // S0/S2 set-up: the ray paths do not change between iterations
    if (rc != LOC_OK) return rc;
    m->ndir = ndir;
    m->ntask = t0;
    return LOC_OK;
}

extern "C" int loc_set_populations(loc_model *m, float *dev_pops)
{
    if (!m || !dev_pops) return LOC_EINVAL;
    if (!m->have_species) return fail(m, LOC_ESTATE, "loc_set_species must be called first");
    m->pops = dev_pops;
    return refresh_coef(m);
}

extern "C" int loc_init_lte(loc_model *m)
{
    if (!m) return LOC_EINVAL;
    if (!m->have_species || !m->pops) return fail(m, LOC_ESTATE, "species and population buffer must be set first");
    int64_t n = m->ncell;
    k_lte<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(n, m->sp, m->cells.density, m->cells.tkin, m->cells.abundance, m->pops);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    return refresh_coef(m);
}

extern "C" int loc_simulate(loc_model *m, int nsel, const int *idx, int geom)
{
    if (!m) return LOC_EINVAL;
    if (!m->have_species || !m->pops) return fail(m, LOC_ESTATE, "species and populations must be set before loc_simulate");
    if (m->kind == LOC_GRID_OCTREE && m->ndir < 1) return fail(m, LOC_ESTATE, "loc_set_directions must be called first");
    if (nsel != 0 || m->selh.nsel == 0) {
        int rc = build_selection(m, nsel, idx);
        if (rc) return rc;
    }
    if (!m->coef_valid) {
        int rc = refresh_coef(m);
        if (rc) return rc;
    }
    int64_t n = m->ncell;
    LOC_CUDA_CHECK(m, cudaMemsetAsync(m->cnt, 0, sizeof(float2) * n * m->selh.nsp, m->stream));
    if (geom) {
        LOC_CUDA_CHECK(m, cudaMemsetAsync(m->visits, 0, sizeof(uint32_t) * n, m->stream));
        LOC_CUDA_CHECK(m, cudaMemsetAsync(m->pathz, 0, sizeof(uint32_t) * n, m->stream));
    }
    LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_steps, 0, 2 * sizeof(unsigned long long), m->stream));
    const int rc = (m->kind == LOC_GRID_SHELL) ? loc_launch_sim1d(m, geom) : loc_launch_sim3d(m, geom);
    m->simulated = rc == LOC_OK;
    return rc;
}

extern "C" int loc_get_counters(loc_model *m, const float **counters, int *ntp, const uint32_t **visits, const uint32_t **pathz)
{
    if (!m) return LOC_EINVAL;
    if (counters) *counters = (const float *)m->cnt;
    if (ntp) *ntp = m->selh.nsp;
    if (visits) *visits = m->visits;
    if (pathz) *pathz = m->pathz;
    return LOC_OK;
}

static int solve_async(loc_model *m)
{
    int64_t n = m->ncell;
    const int32_t *ch = m->kind == LOC_GRID_OCTREE ? m->child : nullptr;
    unsigned nb = (unsigned)((n + 127) / 128);
#define LOC_SOLVE(NLMAX)                                                                                                     \
    k_solve<NLMAX><<<nb, 128, 0, m->stream>>>(n, m->sp, m->selh, m->cells.density, m->cells.tkin, m->cells.abundance, m->cnt, \
                                              m->pops, m->coef, m->d_maxrel, ch, m->ali)
    // shared-memory solver (k_solve_s) while a block's matrices and the species tables fit; loc_set_option(LOC_OPT_SOLVER_LOCAL)
    // forces the local-memory kernel (A/B measurements)
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
        if (NL <= 16 && smem <= 200 * 1024 && !m->solver_local) {
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

static int fetch_maxrel(loc_model *m, double *out)
{
    unsigned int bits = 0;
    int err = 0;
    LOC_CUDA_CHECK(m, cudaMemcpyAsync(&bits, m->d_maxrel, sizeof(bits), cudaMemcpyDeviceToHost, m->stream));
    LOC_CUDA_CHECK(m, cudaMemcpyAsync(&err, m->d_errflag, sizeof(err), cudaMemcpyDeviceToHost, m->stream));
    LOC_CUDA_CHECK(m, cudaStreamSynchronize(m->stream));
    if (err) return fail(m, LOC_ENOMEM, "ray stack overflow inside the traversal kernel");
    float f;
    memcpy(&f, &bits, sizeof(f));
    if (out) *out = f;
    if (!isfinite(f)) return fail(m, LOC_ENONFINITE, "the solve produced a non-finite population (T_kin <= 0, NaN input or counter?)");
    return LOC_OK;
}

extern "C" int loc_solve(loc_model *m, double *max_rel_change)
{
    if (!m) return LOC_EINVAL;
    if (!m->have_species || !m->pops) return fail(m, LOC_ESTATE, "species and populations must be set before loc_solve");
    if (!m->simulated) return fail(m, LOC_ESTATE, "loc_solve: no loc_simulate has filled the counters");
    LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_maxrel, 0, sizeof(unsigned int), m->stream));
    int rc = solve_async(m);
    if (rc) return rc;
    return fetch_maxrel(m, max_rel_change);
}

extern "C" int loc_iterate(loc_model *m, int niter, double *max_rel_change)
{
    if (!m || niter < 0) return LOC_EINVAL;
    if (niter == 0) {  // nothing ran: no stale change of an earlier call
        if (max_rel_change) *max_rel_change = 0.0;
        return LOC_OK;
    }
    for (int it = 0; it < niter; it++) {
        int rc = loc_simulate(m, 0, nullptr, 0);
        if (rc) return rc;
        LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_maxrel, 0, sizeof(unsigned int), m->stream));
        rc = solve_async(m);
        if (rc) return rc;
    }
    return fetch_maxrel(m, max_rel_change);
}

extern "C" int loc_set_ali(loc_model *m, int ali)
{
    if (!m || (ali != 0 && ali != 1)) return LOC_EINVAL;
    m->ali = ali;
    return LOC_OK;
}

extern "C" int loc_set_option(loc_model *m, int key, double value)
{
    if (!m) return LOC_EINVAL;
    switch (key) {
    case LOC_OPT_WINDOW_XMIN:
        if (!(value >= 1.0 && value <= 12.0)) return fail(m, LOC_EINVAL, "LOC_OPT_WINDOW_XMIN must be in [1, 12]");
        m->xmin = (float)value;
        return LOC_OK;
    case LOC_OPT_WINDOW_EPS_TAU:
        if (!(value > 0.0 && value <= 1.0)) return fail(m, LOC_EINVAL, "LOC_OPT_WINDOW_EPS_TAU must be in (0, 1]");
        m->eps_tau = (float)value;
        return LOC_OK;
    case LOC_OPT_SPAN_XCLIP:
        if (!(value >= 1.0 && value <= 12.0)) return fail(m, LOC_EINVAL, "LOC_OPT_SPAN_XCLIP must be in [1, 12]");
        m->xclip = (float)value;
        return LOC_OK;
    case LOC_OPT_SIM3D_PARTS:
        if (!(value >= 0.0 && value <= LOC_MAX_TRANS) || value != floor(value)) return fail(m, LOC_EINVAL, "LOC_OPT_SIM3D_PARTS must be an integer in [0, LOC_MAX_TRANS]");
        m->sim3d_parts = (int)value;
        return LOC_OK;
    case LOC_OPT_SOLVER_LOCAL:
        if (value != 0.0 && value != 1.0) return fail(m, LOC_EINVAL, "LOC_OPT_SOLVER_LOCAL must be 0 or 1");
        m->solver_local = (int)value;
        return LOC_OK;
    }
    return fail(m, LOC_EINVAL, "loc_set_option: unknown key");
}

extern "C" int loc_iterate_until(loc_model *m, int max_iter, double tol, int *niter_done, double *max_rel_change)
{
    if (!m || max_iter < 0 || !(tol >= 0.0)) return LOC_EINVAL;
    double ch = 0.0;
    int it = 0;
    while (it < max_iter) {
        int rc = loc_simulate(m, 0, nullptr, 0);
        if (rc) return rc;
        LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_maxrel, 0, sizeof(unsigned int), m->stream));
        rc = solve_async(m);
        if (rc) return rc;
        rc = fetch_maxrel(m, &ch);  // one host synchronisation per iteration: the stopping rule needs the scalar
        if (rc) return rc;
        it++;
        if (ch <= tol) break;
    }
    if (niter_done) *niter_done = it;
    if (max_rel_change) *max_rel_change = ch;
    return LOC_OK;
}

extern "C" int loc_spectra(loc_model *m, int trans, const double *dir, int nx, int ny, const int64_t *aff, const double *offsets_cm,
                           float *dev_out)
{
    if (!m || !dev_out) return LOC_EINVAL;
    if (!m->have_species || !m->pops) return fail(m, LOC_ESTATE, "species and populations must be set before loc_spectra");
    if (trans < 0 || trans >= m->ntrans || nx < 1 || ny < 1) return fail(m, LOC_EINVAL, "loc_spectra: bad transition or map size");
    return loc_launch_spectra(m, trans, dir, nx, ny, aff, offsets_cm, dev_out);
}

extern "C" int loc_spectra_map(loc_model *m, int trans, const double *dir, int nx, int ny, double pixel_cm, const double *centre_cm,
                               float *dev_out)
{
    if (!m || !dev_out || !dir || !centre_cm) return LOC_EINVAL;
    if (m->kind != LOC_GRID_OCTREE) return fail(m, LOC_ESTATE, "loc_spectra_map: octree models only (shells: loc_spectra with offsets_cm)");
    if (!m->have_species || !m->pops) return fail(m, LOC_ESTATE, "species and populations must be set before loc_spectra_map");
    if (trans < 0 || trans >= m->ntrans || nx < 1 || ny < 1 || !(pixel_cm > 0.0)) return fail(m, LOC_EINVAL, "loc_spectra_map: bad transition, map size or pixel size");
    return loc_launch_spectra_map(m, trans, dir, nx, ny, pixel_cm, centre_cm, dev_out);
}

// T_ex = -(h nu / k) / ln(n_u g_l / (n_l g_u)) per cell (Fig. 4); 0 where the cell holds no molecules
__global__ void k_tex(int64_t n, const float *pop_u, const float *pop_l, double gl_over_gu, double hnu_over_k, const int32_t *child, float *out)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    float t = 0.0f;
    const double nu_ = pop_u[i], nl_ = pop_l[i];
    if (!(child && child[i] >= 0) && nu_ > 0.0 && nl_ > 0.0) t = (float)(-hnu_over_k / log(nu_ * gl_over_gu / nl_));
    out[i] = t;
}

extern "C" int loc_tex(loc_model *m, int trans, float *dev_tex)
{
    if (!m || !dev_tex) return LOC_EINVAL;
    if (!m->have_species || !m->pops) return fail(m, LOC_ESTATE, "species and populations must be set before loc_tex");
    if (trans < 0 || trans >= m->ntrans) return fail(m, LOC_EINVAL, "loc_tex: bad transition");
    const int u = m->h_upper[trans], l = m->h_lower[trans];
    const int64_t n = m->ncell;
    k_tex<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(n, m->pops + (int64_t)u * n, m->pops + (int64_t)l * n, m->h_g[l] / m->h_g[u],
                                                              LOC_HP * m->h_freq[trans] / LOC_KB,
                                                              m->kind == LOC_GRID_OCTREE ? m->child : nullptr, dev_tex);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    return LOC_OK;
}

extern "C" int loc_line_area(loc_model *m, const float *dev_cube, int64_t npix, float *dev_w)
{
    if (!m || npix < 0 || (npix > 0 && (!dev_cube || !dev_w))) return LOC_EINVAL;
    return loc_launch_line_area(m, dev_cube, (long long)npix, dev_w);
}

extern "C" int loc_get_stats(loc_model *m, loc_stats *out)
{
    if (!m || !out) return LOC_EINVAL;
    unsigned long long steps[2] = {0, 0};
    LOC_CUDA_CHECK(m, cudaMemcpyAsync(steps, m->d_steps, sizeof(steps), cudaMemcpyDeviceToHost, m->stream));
    LOC_CUDA_CHECK(m, cudaStreamSynchronize(m->stream));
    out->ncell = m->ncell;
    out->steps = (m->kind == LOC_GRID_SHELL) ? m->steps1d : (int64_t)steps[0];
    out->active_channels = (int64_t)steps[1];
    out->ntrans_sim = m->selh.nsel;
    out->nchannel = m->nch;
    out->kernel_launches = m->launches;
    out->counter_stride = 2 * m->selh.nsp;
    out->setup_steps = m->setup_steps;
    out->setup_ms = m->setup_ms;
    return LOC_OK;
}

extern "C" void loc_destroy_model(loc_model *m)
{
    if (!m) return;
    free(m->h_upper);
    free(m->h_lower);
    free(m->h_A);
    free(m->h_freq);
    free(m->h_rout);
    free(m->h_dirs);
    delete m;
}

extern "C" const char *loc_last_error(const loc_model *m) { return m ? m->err : g_create_err; }
