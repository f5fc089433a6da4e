// loc_internal.cuh -- shared declarations of the CUDA implementation behind include/loc.h.
// Hand-written for sm_100a.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/loc.h"

#define LOC_LB 20              // log2(grid units per root cell)
#define LOC_H0 (1 << LOC_LB)   // grid units per root cell
#define LOC_MAXL LOC_MAX_TREE_LEVELS
#define LOC_MAX_DIRS 65535     // task -> direction table holds 16-bit indices
#define LOC_BUILD_BATCH 262144  // root lines traced per launch of the path builder (16 B x LOC_BUILD_STACK of stack each)
#define LOC_BUILD_STACK 256    // pending rays per root line (PAPER.md:119 estimates ~7*3^(NL-1) stored rays)

// physical constants (CGS, CODATA 2018) -- DESIGN R1
#define LOC_HP 6.62607015e-27
#define LOC_KB 1.380649e-16
#define LOC_CL 2.99792458e10
#define LOC_AMU 1.66053906660e-24
#define LOC_PI 3.14159265358979323846

#define LOC_LOG2E 1.4426950408889634f
#define LOC_XCLIP 3.4f     // 3D kernel: the span reaches at least this many sigma to both sides of the line centre, or the step is masked (default of LOC_OPT_XCLIP)
#define LOC_XFULL 4.8f     // 3D kernel: span + wing extension (or the pair of spans, or the masked window) reach at least this many sigma (default of LOC_OPT_SPAN_XFULL)
#define LOC_THICK_TAU 0.05f   // line-centre optical depth of a step above which exp() is used instead of the series

// ------------------------------------------------------------------------------------------------
// device-side species description (arrays live in the workspace)
// ------------------------------------------------------------------------------------------------
struct SpeciesDev {
    int nlevel, ntrans, ncoll, ntemp;
    const double *energy_K;  // [nlevel]
    const double *g;         // [nlevel]
    const int *upper, *lower;  // [ntrans]
    const double *A;         // [ntrans]
    const double *freq;      // [ntrans]
    const double *bgocc;     // [ntrans] 1/(exp(h nu/k Tbg)-1)
    const int *cu, *cl;      // [ncoll]
    const double *temps;     // [ntemp]
    const double *rates;     // [ntemp][ncoll]
    double mass_amu;
};

// selection of traced transitions: slot k of the per-cell records belongs to transition sel[k]
struct Selection {
    int nsel, nsp;               // nsp = record stride in float2 (nsel padded to even)
    int sel[LOC_MAX_TRANS];
    int upper[LOC_MAX_TRANS], lower[LOC_MAX_TRANS];
    float gratio[LOC_MAX_TRANS]; // g_u/g_l
    float bgocc[LOC_MAX_TRANS];  // background occupation number at the line frequency (Eq. 1 in occupation units)
    double ck[LOC_MAX_TRANS];    // c^3 A / (8 pi nu^3 dv)
};

// hyperfine structure of the traced transitions (loc_set_hyperfine), slot by slot as in Selection: kernel parameter
struct HfsTab {
    int any;                                 // some traced transition has more than one component (or a shifted one)
    int nc[LOC_MAX_TRANS];                   // components of the slot's transition (>= 1)
    float dch[LOC_MAX_TRANS][LOC_MAX_HFS];   // offsets of the components in CHANNELS (dv_k / dv)
    float w[LOC_MAX_TRANS][LOC_MAX_HFS];     // weights
    float lo, hi;                            // smallest / largest offset over all traced transitions, channels
};

// per-direction data of the integer ray lattice (DESIGN 6.3).  Working frame: axis 0 = main axis (zeta), 1 = p, 2 = q;
// axes with a negative direction component are mirrored so that every ray moves towards +zeta, +p, +q.
struct Dir3 {
    int ax[3];              // model axis (0=x,1=y,2=z) of the working axes
    int flip[3];            // per working axis: mirrored?
    unsigned long long T[2];  // fixed-point inverse slopes of p, q: shift(zeta) = floor(zeta 2^32 / T); 0 = zero slope
    unsigned long long M[2];  // floor(2^64 / T): reciprocal for the exact division by multiplication (shift_of)
    int W[3];               // model extent along the working axes in grid units (2^20 per root cell)
    int np, nq;             // root lines along p, q
    float d[3];             // snapped unit propagation direction, model frame
    float sf;               // cm of path per grid unit of zeta = (root_cm / 2^20) / |d_m|
    long long task0;        // index of the direction's first root-line task
};

// one record of the precomputed step stream (8 bytes):  x = cell index (STEP) or slot (SAVE/LOAD)
//   y = dzeta [0..20] | level [21..23] | opcode [24..26]
#define LOC_OP_STEP 0u
#define LOC_OP_BG 1u    // spectrum := background (model boundary / transverse wrap-around)
#define LOC_OP_SAVE 2u  // slot[x] := spectrum   (donor duty at the upstream face of a refined cell)
#define LOC_OP_LOAD 3u  // spectrum := slot[x]   (birth of a ray in a refined region / resume of the donor)
#define LOC_OP_NOP 7u   // padding: every root-ray task is a whole number of LOC_TASK_ALIGN records
#define LOC_TASK_ALIGN 8
#define LOC_REC(op, level, dz) (((unsigned)(op) << 24) | ((unsigned)(level) << 21) | (unsigned)(dz))

struct loc_model {
    int kind;
    cudaStream_t stream;
    char err[512];
    int nch;
    double band_half, dv, tbg;
    int64_t ncell;
    loc_cells cells;
    // workspace carve-up
    char *ws;
    int64_t ws_bytes, ws_used;
    float4 *kin;     // [ncell] vx,vy,vz,sigma_tot
    float2 *coef;    // [ncell][nsp]  (kap, em)
    float2 *cnt;     // [ncell][nsp]  (SJ, ESC)
    uint32_t *visits, *pathz;
    unsigned long long *d_steps;  // [1]
    unsigned int *d_maxrel;       // [1] float bits
    int *d_errflag;               // [1]
    int max_trans, max_levels;    // limits given to loc_create_model
    // species
    bool have_species;
    int nlevel, ntrans, ncoll, ntemp;
    SpeciesDev sp;
    double h_energy[LOC_MAX_LEVELS], h_g[LOC_MAX_LEVELS];
    int *h_upper, *h_lower;
    double *h_A, *h_freq;
    int *h_cu, *h_cl;           // host copies of the collisional pairs, temperatures and rates (dense tables of k_solve_f)
    double *h_temps, *h_rates;
    float *d_rates_f;           // [64][66] dense float32 rate table of k_solve_f (ntemp > 1)
    bool rates_f_valid;
    Selection selh;
    int h_hfs_nc[LOC_MAX_LEVELS * (LOC_MAX_LEVELS - 1) / 2];              // hyperfine components per species transition (0 = none)
    double h_hfs_dv[LOC_MAX_LEVELS * (LOC_MAX_LEVELS - 1) / 2][LOC_MAX_HFS];
    double h_hfs_w[LOC_MAX_LEVELS * (LOC_MAX_LEVELS - 1) / 2][LOC_MAX_HFS];
    bool coef_valid;
    int ali;  // 1: accelerated lambda iteration (default), 0: plain lambda iteration (loc_set_ali)
    float *pops;  // registered [nlevel][ncell]
    // accuracy knobs (DESIGN 5.3), set through loc_set_option only
    float xmin, eps_tau, xclip, xfull;
    int sim3d_parts;   // 0 = automatic split of the traced transitions over launches
    int sim3d_warps;   // 0 = automatic, 1 = one warp per ray set (up to 6 transitions per launch), 2 = two warps
    int solver;        // loc_set_option(LOC_OPT_SOLVER): 0 = automatic, 1 = float64 local memory, 2 = float64 shared memory
    int nsm;           // multiprocessors of the model's device (queried once in loc_create_model)
    bool simulated;    // counters hold the result of a loc_simulate
    // 1D
    int nshell, nray;
    int *d_order, *d_k0;
    long long *d_off;
    float *d_tabs, *d_tabmu, *d_tabw;
    double *h_rout;
    double *d_rout;  // device copy of the shell radii (1D spectra)
    int64_t steps1d;
    // 3D
    int nx, ny, nz, nlev;
    double root_cm;
    int64_t noff[LOC_MAXL + 1];
    const int32_t *child;
    int ndir, ndir_max;
    Dir3 *d_dirs;  // [ndir_max]
    Dir3 *h_dirs;
    unsigned int *d_queue;      // [1] task queue head
    int64_t ntask, ntask_max;
    long long *d_task_off;      // [ntask_max+1] record offsets of the root-line tasks
    uint16_t *d_task_dir;       // [ntask_max] direction of each root-line task (ndir <= LOC_MAX_DIRS)
    uint2 *d_stream;            // precomputed step stream (S0/S2 set-up)
    int64_t stream_cap, stream_len;
    char *d_bstack;             // builder stacks
    int bstack_threads;
    int max_warps;
    float *spec_pool;           // per resident warp: (nlev-1) spectrum slots of [nsel][nch]
    int64_t spec_pool_floats;
    int64_t setup_steps;
    double setup_ms;
    // stats
    int64_t launches;
};

// ------------------------------------------------------------------------------------------------
// device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2f(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Packed float32 pairs (sm_100a `*.f32x2`): one instruction updates two channels.  On B200 an FFMA2 holds the FMA pipe
// for two cycles like two FFMA, but takes ONE issue slot (measured: profiles/r1_pipe_microbench.md) -- the 3D kernel is
// issue bound, so the bulk per-channel arithmetic is written in pairs.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// Per-transition parameters of one ray step, computed once per (step, transition)
struct __align__(16) TParam {
    float c0;     // thick: -kap*s*log2(e)      thin: kap*s
    float c1;     // thick: em/kap (source)     thin: em*s
    float scale;  // thick: w/(kap*s)           thin: w       multiplies the channel sums
    int thick;
};

__device__ __forceinline__ TParam make_tparam(float2 ke, float s, float w, float amp)
{
    TParam p;
    float ks = ke.x * s;
    bool thick = fabsf(ks) * amp >= LOC_THICK_TAU;
    if (thick) {
        float inv = __fdividef(1.0f, ke.x);
        p.c0 = -ks * LOC_LOG2E;
        p.c1 = ke.y * inv;
        p.scale = __fdividef(w, ks);
    } else {
        p.c0 = ks;
        p.c1 = ke.y * s;
        p.scale = w;
    }
    p.thick = thick;
    return p;
}

// One channel, one transition (Eq. 3 and the two sums of Eq. 2 / PAPER.md:81 in occupation-number units):
//   n      photon occupation number in the channel, updated
//   phi    fraction of the profile in the channel (0 for inactive lanes)
//   accA  += n_in * phi * f(tau)        (thick: n_in (1-e^-tau), rescaled by 1/(kap s) afterwards)
//   accB  += phi * f(tau)               (thick: (1-e^-tau))
// The same for a quad of channels in packed pairs (half the issue slots).  n01 / n23 and phi01 / phi23 hold channels (0, 1) / (2, 3); acc += the quad's sums.
__device__ __forceinline__ void channel_update4(f32x2 &n01, f32x2 &n23, f32x2 phi01, f32x2 phi23, const TParam &p, float &accA, float &accB)
{
    const f32x2 C0 = pk2(p.c0, p.c0), C1 = pk2(p.c1, p.c1);
    const f32x2 ONE = pk2(1.0f, 1.0f), MONE = pk2(-1.0f, -1.0f);
    float a0, a1, b0, b1;
    if (p.thick) {
        float z0, z1, z2, z3;
        upk2(mul2(phi01, C0), z0, z1);
        upk2(mul2(phi23, C0), z2, z3);
        const f32x2 om01 = fma2(pk2(ex2f(z0), ex2f(z1)), MONE, ONE), om23 = fma2(pk2(ex2f(z2), ex2f(z3)), MONE, ONE);
        upk2(fma2(n01, om01, mul2(n23, om23)), a0, a1);
        upk2(add2(om01, om23), b0, b1);
        n01 = fma2(om01, fma2(n01, MONE, C1), n01);
        n23 = fma2(om23, fma2(n23, MONE, C1), n23);
    } else {
        const f32x2 K4 = pk2(-1.0f / 24.0f, -1.0f / 24.0f), K3 = pk2(1.0f / 6.0f, 1.0f / 6.0f), K2 = pk2(-0.5f, -0.5f);
        const f32x2 t01 = mul2(phi01, C0), t23 = mul2(phi23, C0);
        const f32x2 P01 = fma2(t01, fma2(t01, fma2(t01, K4, K3), K2), ONE), P23 = fma2(t23, fma2(t23, fma2(t23, K4, K3), K2), ONE);
        const f32x2 q01 = mul2(phi01, P01), q23 = mul2(phi23, P23);
        const f32x2 om01 = mul2(t01, P01), om23 = mul2(t23, P23);
        upk2(fma2(n01, q01, mul2(n23, q23)), a0, a1);
        upk2(add2(q01, q23), b0, b1);
        n01 = fma2(C1, q01, fma2(mul2(n01, MONE), om01, n01));
        n23 = fma2(C1, q23, fma2(mul2(n23, MONE), om23, n23));
    }
    accA += a0 + a1;
    accB += b0 + b1;
}

// Reduce NV per-lane values across the warp with a halving butterfly (about NV shuffles in total instead of
// 5 NV).  On return v[0] of lane L holds the warp total of value index *owner (or *owner = -1); every value index has
// exactly one owner lane.
template <int N, int OFF>
struct MultiReduce {
    __device__ static __forceinline__ void run(float *v, int lane, int &base, int &nvalid)
    {
        constexpr int C = (N + 1) / 2;  // kept by the lower half
        constexpr int Hh = N - C;       // kept by the upper half
        const bool up = lane & OFF;
#pragma unroll
        for (int i = 0; i < C; i++) {
            if (i < Hh) {
                float keep = up ? v[i + C] : v[i];
                float send = up ? v[i] : v[i + C];
                v[i] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
            } else {  // unpaired middle value: lower half keeps it, upper half's copy becomes junk
                float other = __shfl_xor_sync(0xffffffffu, v[i], OFF);
                v[i] = up ? 0.0f : v[i] + other;
            }
        }
        if (up) {
            base += C;
            nvalid = max(0, nvalid - C);
        } else {
            nvalid = min(nvalid, C);
        }
        if constexpr (OFF > 1) MultiReduce<C, OFF / 2>::run(v, lane, base, nvalid);
    }
};
template <int OFF>
struct MultiReduce<1, OFF> {
    __device__ static __forceinline__ void run(float *v, int lane, int &base, int &nvalid)
    {
        // a single value left: plain butterfly over the remaining offsets
#pragma unroll
        for (int o = OFF; o >= 1; o >>= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], o);
        if (lane & (2 * OFF - 1)) nvalid = 0;  // the 2*OFF lanes of the group hold copies: only the first one owns the total
    }
};

template <int NV>
__device__ __forceinline__ float warp_multi_reduce(float (&v)[NV], int lane, int &owner)
{
    int base = 0, nvalid = NV;
    MultiReduce<NV, 16>::run(v, lane, base, nvalid);
    owner = (nvalid >= 1) ? base : -1;
    return v[0];
}

// ------------------------------------------------------------------------------------------------
// integer lattice helpers (device)
// ------------------------------------------------------------------------------------------------
struct Tree {
    int nx, ny, nz, nlev;
    long long noff[LOC_MAXL + 1];
    const int32_t *child;
};

#define LOC_ZINF (1ll << 40)

// floor(z 2^32 / T), exactly, without a 64-bit division (about 100 instructions, several per ray step in the path
// builder): q' = mulhi(n, M) with M = floor(2^64 / T) satisfies q - 1 <= q' <= q for n = z 2^32 < 2^63 and T >= 2^32
// (n (2^64/T - M) / 2^64 < 1), so one remainder test makes it exact; the loop form costs nothing and needs no such bound.
__device__ __forceinline__ long long shift_of(const Dir3 &D, int k, long long z)
{
    const unsigned long long T = D.T[k];
    if (T == 0) return 0ll;
    const unsigned long long n = (unsigned long long)z << 32;
    unsigned long long q = __umul64hi(n, D.M[k]);
    unsigned long long r = n - q * T;
    while (r >= T) {
        r -= T;
        q++;
    }
    return (long long)q;
}

// a / W and a - (a / W) W (floor division) for a that lies within a few W of [0, W): the transverse wrap-around count
__device__ __forceinline__ long long wrap_of(long long a, long long W, long long &rem)
{
    if (a >= 8 * W || a < -8 * W) {
        const long long w = (a >= 0) ? a / W : -((-a + W - 1) / W);
        rem = a - w * W;
        return w;
    }
    long long w = 0;
    while (a >= W) {
        a -= W;
        w++;
    }
    while (a < 0) {
        a += W;
        w--;
    }
    rem = a;
    return w;
}

// smallest zeta with shift_of(T, zeta) >= D
__device__ __forceinline__ long long cross_of(unsigned long long T, long long D)
{
    if (D <= 0) return 0;
    if (T == 0) return LOC_ZINF;
    unsigned long long lo = (unsigned long long)D * T, hi = __umul64hi((unsigned long long)D, T);
    unsigned long long lo2 = lo + 0xffffffffull;
    if (lo2 < lo) hi++;
    return (long long)((hi << 32) | (lo2 >> 32));
}


struct LeafPos {
    int cell[LOC_MAXL];  // global cell index of the ancestor at each level (last = the leaf)
    int level;
};

// leaf containing the working-frame point (fz, fp, fq), all coordinates inside the model
__device__ __forceinline__ void find_leaf(const Tree &G, const Dir3 &D, int fz, int fp, int fq, LeafPos &L)
{
    int X[3];
    X[D.ax[0]] = D.flip[0] ? D.W[0] - 1 - fz : fz;
    X[D.ax[1]] = D.flip[1] ? D.W[1] - 1 - fp : fp;
    X[D.ax[2]] = D.flip[2] ? D.W[2] - 1 - fq : fq;
    int g = (X[0] >> LOC_LB) + G.nx * ((X[1] >> LOC_LB) + G.ny * (X[2] >> LOC_LB));
    int l = 0;
    L.cell[0] = g;
    int ch;
    while ((ch = __ldg(G.child + g)) >= 0) {
        int bit = LOC_LB - 1 - l;
        g = (int)G.noff[l + 1] + ch + ((X[0] >> bit) & 1) + 2 * ((X[1] >> bit) & 1) + 4 * ((X[2] >> bit) & 1);
        l++;
        L.cell[l] = g;
    }
    L.level = l;
}

__device__ __forceinline__ int level_at(const Tree &G, const Dir3 &D, int fz, int fp, int fq)
{
    LeafPos L;
    find_leaf(G, D, fz, fp, fq, L);
    return L.level;
}

static inline Tree make_tree(const loc_model *m)
{
    Tree G;
    G.nx = m->nx;
    G.ny = m->ny;
    G.nz = m->nz;
    G.nlev = m->nlev;
    for (int l = 0; l <= LOC_MAXL; l++) G.noff[l] = (l <= m->nlev) ? m->noff[l] : m->noff[m->nlev];
    G.child = m->child;
    return G;
}

// ------------------------------------------------------------------------------------------------
// kernels / launchers implemented in the other translation units
// ------------------------------------------------------------------------------------------------
int loc_launch_solve(loc_model *m);
void loc_fill_hfs(const loc_model *m, HfsTab &H);                       // table of the current selection
void loc_fill_hfs_one(const loc_model *m, int trans, HfsTab &H);        // slot 0 = species transition `trans` (spectra)
int loc_launch_sim1d(loc_model *m, int geom);
int loc_launch_sim3d(loc_model *m, int geom);
int loc_setup3d(loc_model *m);
int loc_launch_spectra(loc_model *m, int trans, const double *dir, int nx, int ny, const int64_t *aff,
                       const double *offsets_cm, float *dev_out);
int loc_launch_spectra_map(loc_model *m, int trans, const double *dir, int nx, int ny, double pixel_cm, const double *centre_cm,
                           float *dev_out);
int loc_launch_line_area(loc_model *m, const float *dev_cube, long long npix, float *dev_w);
int loc_build_streams(loc_model *m, int ndir, int64_t ntask);
void loc_fill_dir(loc_model *m, const double *din, Dir3 *D);

#define LOC_CUDA_CHECK(m, call)                                                                    \
    do {                                                                                           \
        cudaError_t _e = (call);                                                                   \
        if (_e != cudaSuccess) {                                                                   \
            snprintf((m)->err, sizeof((m)->err), "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(_e)); \
            return LOC_ECUDA;                                                                      \
        }                                                                                          \
    } while (0)
