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

static thread_local char g_create_err[512] = "";  // per thread: loc_create_model has no model to carry its error text

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
// upper bound used to size the per-CTA spectrum slots of k_sim3d: 32 CTAs per multiprocessor is the hardware's limit, so the
// launch (occupancy query x multiprocessors) is never clamped by the pool whatever a kernel variant's register / shared-
// memory use allows (round 2 sized it for 16: right for today's 128-register one-warp CTAs, a silent cap for leaner ones)
static int max_resident_ctas() { return device_sm_count() * 32; }

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
    m->d_rates_f = c.take<float>(64 * 66);
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
    for (int k = nsel; k < LOC_MAX_TRANS; k++) S.bgocc[k] = 0.0f;  // (pad slots of the 3D kernel: no photons)
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
    m->xfull = LOC_XFULL;
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
    for (int j = 1; temps_K && j < ntemp; j++)
        if (!(temps_K[j] > temps_K[j - 1])) return fail(m, LOC_EINVAL, "collision temperatures must ascend");
    m->nlevel = nlevel;
    m->ntrans = ntrans;
    m->ncoll = ncoll;
    m->ntemp = ntemp;
    memcpy(m->h_energy, energy_K, sizeof(double) * nlevel);
    memcpy(m->h_g, g, sizeof(double) * nlevel);
    free(m->h_upper); free(m->h_lower); free(m->h_A); free(m->h_freq);
    free(m->h_cu); free(m->h_cl); free(m->h_temps); free(m->h_rates);
    m->have_species = false;
    m->simulated = false;  // counters traced for the previous species say nothing about this one
    m->h_cu = (int *)calloc(std::max(ncoll, 1), sizeof(int));
    m->h_cl = (int *)calloc(std::max(ncoll, 1), sizeof(int));
    m->h_temps = (double *)calloc(ntemp, sizeof(double));
    m->h_rates = (double *)calloc((size_t)ntemp * std::max(ncoll, 1), sizeof(double));
    m->h_upper = (int *)calloc(ntrans, sizeof(int));
    m->h_lower = (int *)calloc(ntrans, sizeof(int));
    m->h_A = (double *)calloc(ntrans, sizeof(double));
    m->h_freq = (double *)calloc(ntrans, sizeof(double));
    if (!m->h_cu || !m->h_cl || !m->h_temps || !m->h_rates || !m->h_upper || !m->h_lower || !m->h_A || !m->h_freq)
        return fail(m, LOC_ENOMEM, "loc_set_species: host allocation failed");
    // a species without collisions may still carry a temperature grid (ntemp > 1): the solvers interpolate on it
    if (temps_K) memcpy(m->h_temps, temps_K, sizeof(double) * ntemp);
    else for (int j = 0; j < ntemp; j++) m->h_temps[j] = 1.0 + j;
    if (ncoll) {
        memcpy(m->h_cu, cu, sizeof(int) * ncoll);
        memcpy(m->h_cl, cl, sizeof(int) * ncoll);
        memcpy(m->h_rates, rate_down, sizeof(double) * ntemp * ncoll);
    }
    m->rates_f_valid = false;
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
    LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.temps, m->h_temps, sizeof(double) * ntemp, cudaMemcpyHostToDevice, st));
    if (ncoll) {
        LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.cu, cu, sizeof(int) * ncoll, cudaMemcpyHostToDevice, st));
        LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.cl, cl, sizeof(int) * ncoll, cudaMemcpyHostToDevice, st));
        LOC_CUDA_CHECK(m, cudaMemcpyAsync((void *)sp.rates, rate_down, sizeof(double) * ntemp * ncoll, cudaMemcpyHostToDevice, st));
    }
    m->have_species = true;
    {
        int rc = loc_refresh_cells(m);
        if (rc) return rc;
    }
    LOC_CUDA_CHECK(m, cudaStreamSynchronize(st));  // bg vector goes out of scope
    m->have_species = true;
    memset(m->h_hfs_nc, 0, sizeof(m->h_hfs_nc));  // a new species has no hyperfine structure until loc_set_hyperfine
    m->selh.nsel = 0;
    m->coef_valid = false;
    return build_selection(m, 0, nullptr);
}

static void fill_hfs_slot(const loc_model *m, int t, int k, HfsTab &H)
{
    const int nc = m->h_hfs_nc[t];
    H.nc[k] = nc > 0 ? nc : 1;
    for (int c = 0; c < LOC_MAX_HFS; c++) {
        H.dch[k][c] = (nc > 0 && c < nc) ? (float)(m->h_hfs_dv[t][c] / m->dv) : 0.0f;
        H.w[k][c] = (nc > 0) ? (c < nc ? (float)m->h_hfs_w[t][c] : 0.0f) : (c == 0 ? 1.0f : 0.0f);
    }
    for (int c = 0; c < H.nc[k]; c++) {
        H.lo = std::min(H.lo, H.dch[k][c]);
        H.hi = std::max(H.hi, H.dch[k][c]);
        if (H.dch[k][c] != 0.0f || H.nc[k] > 1) H.any = 1;
    }
}

void loc_fill_hfs(const loc_model *m, HfsTab &H)
{
    memset(&H, 0, sizeof(H));
    for (int k = 0; k < m->selh.nsel; k++) fill_hfs_slot(m, m->selh.sel[k], k, H);
}

void loc_fill_hfs_one(const loc_model *m, int trans, HfsTab &H)
{
    memset(&H, 0, sizeof(H));
    fill_hfs_slot(m, trans, 0, H);
}

extern "C" int loc_set_hyperfine(loc_model *m, int trans, int ncomp, const double *dv_cm_s, const double *weight)
{
    if (!m) return LOC_EINVAL;
    if (!m->have_species) return fail(m, LOC_ESTATE, "loc_set_species must be called before loc_set_hyperfine");
    if (trans < 0 || trans >= m->ntrans) return fail(m, LOC_EINVAL, "loc_set_hyperfine: transition index out of range");
    if (ncomp < 0 || ncomp > LOC_MAX_HFS || (ncomp > 0 && (!dv_cm_s || !weight))) return fail(m, LOC_EINVAL, "loc_set_hyperfine: ncomp must be in [0, LOC_MAX_HFS]");
    double sum = 0.0;
    for (int k = 0; k < ncomp; k++) {
        if (!(weight[k] > 0.0) || !(fabs(dv_cm_s[k]) <= 2.0 * m->band_half)) return fail(m, LOC_EINVAL, "loc_set_hyperfine: weights must be > 0 and offsets within the band width");
        sum += weight[k];
    }
    if (ncomp > 0 && fabs(sum - 1.0) > 1e-6) return fail(m, LOC_EINVAL, "loc_set_hyperfine: the weights must sum to 1");
    m->simulated = false;  // the counters were traced with the old profile
    m->h_hfs_nc[trans] = ncomp;
    for (int k = 0; k < ncomp; k++) {
        m->h_hfs_dv[trans][k] = dv_cm_s[k];
        m->h_hfs_w[trans][k] = weight[k];
    }
    return LOC_OK;
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
    int rc = loc_launch_solve(m);
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
        rc = loc_launch_solve(m);
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
    case LOC_OPT_SPAN_XFULL:
        if (!(value >= 1.0 && value <= 12.0)) return fail(m, LOC_EINVAL, "LOC_OPT_SPAN_XFULL must be in [1, 12]");
        m->xfull = (float)value;
        return LOC_OK;
    case LOC_OPT_SIM3D_WARPS:
        if (value != 0.0 && value != 1.0 && value != 2.0) return fail(m, LOC_EINVAL, "LOC_OPT_SIM3D_WARPS must be 0, 1 or 2");
        m->sim3d_warps = (int)value;
        return LOC_OK;
    case LOC_OPT_SOLVER:
        if (value != 0.0 && value != 1.0 && value != 2.0) return fail(m, LOC_EINVAL, "LOC_OPT_SOLVER must be 0, 1 or 2");
        m->solver = (int)value;
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
        rc = loc_launch_solve(m);
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
    out->active_updates = (int64_t)steps[1];
    out->active_channels = m->selh.nsel > 0 ? (int64_t)steps[1] / m->selh.nsel : 0;
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
    free(m->h_cu);
    free(m->h_cl);
    free(m->h_temps);
    free(m->h_rates);
    free(m->h_rout);
    free(m->h_dirs);
    delete m;
}

extern "C" const char *loc_last_error(const loc_model *m) { return m ? m->err : g_create_err; }
