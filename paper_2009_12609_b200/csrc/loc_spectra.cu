// loc_spectra.cu -- spectral-line map kernels (S10; "spectral line maps ... are calculated for selected
// transitions by a final line-of-sight integration through the model", "simple tracing of individual rays
// through an octree", PAPER.md:203 pixel = smallest cell).
//
// Octree maps: a quarter-warp per line of sight (map pixel), four neighbouring pixels per warp; shell models: one warp per
// line of sight.  The pixel's spectrum lives in shared memory as the EXCESS photon occupation
// number over the background, D_c = n_c - n_bg, so that the output T_A(c) = (h nu / k) D_c (= (c^2/2k nu^2)(I_c - B_nu(T_bg)))
// carries no cancellation:
//     D_c <- D_c + X_c (S - n_bg - D_c),   X_c = 1 - exp(-tau_c),   tau_c = kap s phi_c,   S = n_u / (n_l g_u/g_l - n_u)
// (the formal solution I <- I e^-tau + S_nu (1 - e^-tau) in occupation-number units, DESIGN 5.2).  The path is walked by all
// lanes of a line of sight in lock step with the integer lattice arithmetic of the path builder (DESIGN R7) -- no births, no wrap-around: a line
// of sight starts where it enters the model and ends where it leaves it -- and the lanes then split the channels of the
// step's profile window (DESIGN R13).  kap and S are formed in double from the float32 populations (n_l g_u/g_l - n_u cancels).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>

#include "loc_internal.cuh"

#define LOC_SPEC_WARPS 4       // lines of sight per block
#define LOC_SPEC_BATCH1D 256   // 1D lines of sight per launch (their impact parameters travel as kernel arguments)

struct SpecCommon {
    int nch, nchp;
    float dv, xmin;
    float tk_per_occ;  // h nu / k: antenna temperature per unit of occupation number
    float bgocc;       // background occupation number at the line frequency
    double ck, gratio; // c^3 A / (8 pi nu^3 dv), g_u / g_l
    int64_t ncell;
    const float *pop_u, *pop_l;
    const float4 *kin;
    float *out;
    // hyperfine structure of the transition (loc_set_hyperfine): nc components at dch channels from the line centre
    int nc;
    float dch[LOC_MAX_HFS], wgt[LOC_MAX_HFS], lo, hi;
};

// one cell step of a line of sight: the LPL lanes that carry it split the channels of the window (lane l owns the channels
// c = l mod LPL throughout, so the lanes of a line of sight never touch each other's channels: no synchronisation)
template <int LPL>
__device__ __forceinline__ void spectrum_step(const SpecCommon &C, float *D, int lane, long long cell, float s, float v0, float sig)
{
    const double nu_ = (double)__ldg(C.pop_u + cell), nl_ = (double)__ldg(C.pop_l + cell);
    const double den = nl_ * C.gratio - nu_;
    if (den == 0.0) return;  // no molecules (or exactly saturated): tau = 0
    const float kap = (float)(C.ck * den);
    const float src = (float)(nu_ / den) - C.bgocc;
    const float inv_sig = __fdividef(1.0f, sig);
    const float amp = C.dv * 0.3989422804f * inv_sig;
    const float ks = kap * s;
    const float tau0 = fabsf(ks) * amp;
    float X = C.xmin;
    if (tau0 > 1.0f) X = sqrtf(fmaf(2.0f, __logf(tau0), X * X));
    const float inv_dv = __fdividef(1.0f, C.dv);
    const float cc = fmaf(v0, inv_dv, 0.5f * (float)(C.nch - 1));
    const float hw = X * sig * inv_dv;
    const int clo = max(0, (int)ceilf(cc + C.lo - hw)), chi = min(C.nch - 1, (int)floorf(cc + C.hi + hw));
    const float ky = C.dv * 0.8493218f * inv_sig, lamp = __log2f(amp);
    const bool thick = tau0 >= 0.03f;
    for (int c = clo + ((lane - clo) & (LPL - 1)); c <= chi; c += LPL) {
        float phi;
        if (C.nc == 1 && C.dch[0] == 0.0f) {
            const float y = ((float)c - cc) * ky;
            phi = ex2f(fmaf(-y, y, lamp));
        } else {  // sum over the hyperfine components (LTE between them, one source function)
            phi = 0.0f;
            for (int q = 0; q < C.nc; q++) {
                const float y = ((float)c - cc - C.dch[q]) * ky;
                phi = fmaf(C.wgt[q], ex2f(fmaf(-y, y, lamp)), phi);
            }
        }
        const float tau = ks * phi;
        float Xc;
        if (thick)
            Xc = 1.0f - ex2f(-tau * LOC_LOG2E);
        else
            Xc = tau * fmaf(tau, fmaf(tau, fmaf(tau, -1.0f / 24.0f, 1.0f / 6.0f), -0.5f), 1.0f);
        const float d = D[c];
        D[c] = fmaf(Xc, src - d, d);
    }
}

struct Spec3D {
    SpecCommon C;
    Tree G;
    Dir3 D;
    int nx, ny;
    // pixel (ix, iy) starts on the upstream face at the working-frame transverse position
    //   floor((o[0] + ix ex[0]) + iy ey[0]),  floor((o[1] + ix ex[1]) + iy ey[1])      (grid units, 2^20 per root cell),
    // each product and sum rounded to nearest double on its own (no FMA contraction), so that a caller can reproduce the
    // positions bit for bit; with integer coefficients (loc_spectra's `aff`) every term is exact
    double o[2], ex[2], ey[2];
};

// Octree: a quarter-warp per line of sight, four neighbouring pixels per warp (round 1 gave a whole warp to each: all 32
// lanes repeated the 64-bit lattice walk and the ~40 channels of a step's window left the second trip over the lanes
// mostly idle: C5 cube 143 ms).  The four walks of a warp diverge only where their cells differ in refinement.
#define LOC_SPEC_LPL 8
__global__ void __launch_bounds__(32 * LOC_SPEC_WARPS) k_spectra3d(Spec3D P)
{
    extern __shared__ __align__(16) float smem[];
    constexpr int LPW = 32 / LOC_SPEC_LPL;  // lines of sight per warp
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, grp = lane / LOC_SPEC_LPL, l = lane % LOC_SPEC_LPL;
    const long long pix = ((long long)blockIdx.x * LOC_SPEC_WARPS + warp) * LPW + grp;
    if (pix >= (long long)P.nx * P.ny) return;
    float *Dc = smem + (warp * LPW + grp) * P.C.nchp;
    for (int c = l; c < P.C.nchp; c += LOC_SPEC_LPL) Dc[c] = 0.f;
    const int ix = (int)(pix % P.nx), iy = (int)(pix / P.nx);
    const long long bp = (long long)floor(__dadd_rn(__dadd_rn(P.o[0], __dmul_rn((double)ix, P.ex[0])), __dmul_rn((double)iy, P.ey[0])));
    const long long bq = (long long)floor(__dadd_rn(__dadd_rn(P.o[1], __dmul_rn((double)ix, P.ex[1])), __dmul_rn((double)iy, P.ey[1])));
    const Dir3 &D = P.D;
    const long long Wz = D.W[0], Wp = D.W[1], Wq = D.W[2];
    long long zeta = 0;
    // a line that starts beside the model enters through a side face: advance to the first zeta at which it is inside
    if (bp < 0) zeta = max(zeta, cross_of(D.T[0], -bp));
    if (bq < 0) zeta = max(zeta, cross_of(D.T[1], -bq));
    while (zeta < Wz) {
        const long long up = bp + shift_of(D, 0, zeta), uq = bq + shift_of(D, 1, zeta);
        if (up < 0 || uq < 0 || up >= Wp || uq >= Wq) break;  // left through a side face
        LeafPos L;
        find_leaf(P.G, D, (int)zeta, (int)up, (int)uq, L);
        const long long h = LOC_H0 >> L.level;
        long long znext = (zeta & ~(h - 1)) + h, z;
        z = cross_of(D.T[0], (up & ~(h - 1)) + h - bp); if (z < znext) znext = z;
        z = cross_of(D.T[1], (uq & ~(h - 1)) + h - bq); if (z < znext) znext = z;
        const long long cell = L.cell[L.level];
        const float4 k = __ldg(P.C.kin + cell);
        const float v0 = -(k.x * D.d[0] + k.y * D.d[1] + k.z * D.d[2]);  // DESIGN R6
        spectrum_step<LOC_SPEC_LPL>(P.C, Dc, l, cell, (float)(znext - zeta) * D.sf, v0, k.w);
        zeta = znext;
    }
    float *o = P.C.out + pix * P.C.nch;
    for (int c = l; c < P.C.nch; c += LOC_SPEC_LPL) o[c] = P.C.tk_per_occ * Dc[c];
}

struct Spec1D {
    SpecCommon C;
    int ns, nlos;
    const double *r_out;  // device [ns]
    double b[LOC_SPEC_BATCH1D];
};

// 1D: line of sight at impact parameter b through the shells: in through NS-1 .. k0+1, the tangent shell k0 as one step
// (DESIGN R5), out through k0+1 .. NS-1; Doppler shift from the direction cosine at the ENTRY of each step.
__global__ void __launch_bounds__(32 * LOC_SPEC_WARPS) k_spectra1d(Spec1D P)
{
    extern __shared__ __align__(16) float smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int los = blockIdx.x * LOC_SPEC_WARPS + warp;
    if (los >= P.nlos) return;
    float *Dc = smem + warp * P.C.nchp;
    for (int c = lane; c < P.C.nchp; c += 32) Dc[c] = 0.f;
    __syncwarp();
    const double b = fabs(P.b[los]);
    const int ns = P.ns;
    if (b < P.r_out[ns - 1]) {
        int k0 = 0;
        while (k0 < ns - 1 && b >= P.r_out[k0]) k0++;
        const double b2 = b * b;
        for (int j = 0; j < 2 * (ns - 1 - k0) + 1; j++) {
            const int nin = ns - 1 - k0;
            const int k = (j < nin) ? ns - 1 - j : k0 + (j - nin);
            const double ro = P.r_out[k], ri = (k > 0) ? P.r_out[k - 1] : 0.0;
            double s, mu;
            if (j < nin) {
                s = sqrt(ro * ro - b2) - sqrt(ri * ri - b2);
                mu = -sqrt(1.0 - b2 / (ro * ro));
            } else if (j == nin) {
                s = 2.0 * sqrt(ro * ro - b2);
                mu = -sqrt(1.0 - b2 / (ro * ro));
            } else {
                s = sqrt(ro * ro - b2) - sqrt(ri * ri - b2);
                mu = sqrt(1.0 - b2 / (ri * ri));
            }
            const float4 kk = __ldg(P.C.kin + k);
            spectrum_step<32>(P.C, Dc, lane, k, (float)s, -kk.x * (float)mu, kk.w);
        }
    }
    __syncwarp();
    float *o = P.C.out + (long long)los * P.C.nch;
    for (int c = lane; c < P.C.nch; c += 32) o[c] = P.C.tk_per_occ * Dc[c];
}

static void spec_common(loc_model *m, int trans, SpecCommon &C)
{
    const int u = m->h_upper[trans], l = m->h_lower[trans];
    const double nu = m->h_freq[trans];
    C.nch = m->nch;
    C.nchp = (m->nch + 3) & ~3;
    C.dv = (float)m->dv;
    C.xmin = 6.0f;  // wider than the simulation's window: the map is cheap, and tau_edge = e^-18 tau-independent (DESIGN R13)
    C.tk_per_occ = (float)(LOC_HP * nu / LOC_KB);
    C.bgocc = (m->tbg > 0.0) ? (float)(1.0 / expm1(LOC_HP * nu / (LOC_KB * m->tbg))) : 0.0f;
    C.ck = LOC_CL * LOC_CL * LOC_CL * m->h_A[trans] / (8.0 * LOC_PI * nu * nu * nu * m->dv);
    C.gratio = m->h_g[u] / m->h_g[l];
    C.ncell = m->ncell;
    C.pop_u = m->pops + (int64_t)u * m->ncell;
    C.pop_l = m->pops + (int64_t)l * m->ncell;
    C.kin = m->kin;
    HfsTab H;
    loc_fill_hfs_one(m, trans, H);
    C.nc = H.nc[0];
    for (int q = 0; q < LOC_MAX_HFS; q++) {
        C.dch[q] = H.dch[0][q];
        C.wgt[q] = H.w[0][q];
    }
    C.lo = H.lo;
    C.hi = H.hi;
}

static int launch_spectra3d(loc_model *m, int trans, const double *dir, int nx, int ny, const double *o, const double *ex, const double *ey,
                            float *dev_out)
{
    const double nn = dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2];
    if (!(fabs(nn - 1.0) < 1e-9)) {
        snprintf(m->err, sizeof(m->err), "loc_spectra: direction is not a unit vector");
        return LOC_EINVAL;
    }
    Spec3D P;
    spec_common(m, trans, P.C);
    P.C.out = dev_out;
    P.G = make_tree(m);
    loc_fill_dir(m, dir, &P.D);
    P.nx = nx;
    P.ny = ny;
    for (int i = 0; i < 2; i++) {
        P.o[i] = o[i];
        P.ex[i] = ex[i];
        P.ey[i] = ey[i];
    }
    constexpr int PPB = LOC_SPEC_WARPS * (32 / LOC_SPEC_LPL);  // pixels per block
    const size_t smem = sizeof(float) * PPB * P.C.nchp;
    const long long npix = (long long)nx * ny;
    if (smem > 48 * 1024) LOC_CUDA_CHECK(m, cudaFuncSetAttribute(k_spectra3d, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_spectra3d<<<(unsigned)((npix + PPB - 1) / PPB), 32 * LOC_SPEC_WARPS, smem, m->stream>>>(P);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    return LOC_OK;
}

int loc_launch_spectra(loc_model *m, int trans, const double *dir, int nx, int ny, const int64_t *aff, const double *offsets_cm,
                       float *dev_out)
{
    if (m->kind == LOC_GRID_OCTREE) {
        if (!dir || !aff) {
            snprintf(m->err, sizeof(m->err), "loc_spectra: octree models need dir and aff");
            return LOC_EINVAL;
        }
        const double o[2] = {(double)aff[0], (double)aff[1]}, ex[2] = {(double)aff[2], (double)aff[4]}, ey[2] = {(double)aff[3], (double)aff[5]};
        return launch_spectra3d(m, trans, dir, nx, ny, o, ex, ey, dev_out);
    }
    if (ny != 1 || !offsets_cm) {
        snprintf(m->err, sizeof(m->err), "loc_spectra: shell models need ny = 1 and offsets_cm");
        return LOC_EINVAL;
    }
    SpecCommon C;
    spec_common(m, trans, C);
    const size_t smem = sizeof(float) * LOC_SPEC_WARPS * C.nchp;
    for (int b0 = 0; b0 < nx; b0 += LOC_SPEC_BATCH1D) {
        Spec1D P;
        P.C = C;
        P.C.out = dev_out + (int64_t)b0 * m->nch;
        P.ns = m->nshell;
        P.nlos = std::min(nx - b0, LOC_SPEC_BATCH1D);
        P.r_out = m->d_rout;
        for (int i = 0; i < LOC_SPEC_BATCH1D; i++) P.b[i] = (i < P.nlos) ? offsets_cm[b0 + i] : 0.0;
        k_spectra1d<<<(P.nlos + LOC_SPEC_WARPS - 1) / LOC_SPEC_WARPS, 32 * LOC_SPEC_WARPS, smem, m->stream>>>(P);
        m->launches++;
        LOC_CUDA_CHECK(m, cudaGetLastError());
    }
    return LOC_OK;
}

// Map in the caller's frame (include/loc.h, loc_spectra_map): the image plane is spanned by e2 = the unit projection of
// "north" (z; y when dir is parallel to z) perpendicular to dir and e1 = e2 x dir; pixel (ix, iy) is the line of sight through
// X = centre + (ix - (nx-1)/2) pixel e1 + (iy - (ny-1)/2) pixel e2.  In the working frame of the direction (main axis zeta,
// transverse p, q, mirrored so that the ray moves towards + on all three) the line is at p(zeta) = p_X + s_p (zeta - zeta_X),
// s_p the snapped slope 2^32 / T; its start on the upstream face zeta = 0 is an affine function of (ix, iy).
int loc_launch_spectra_map(loc_model *m, int trans, const double *dir, int nx, int ny, double pixel_cm, const double *centre_cm,
                           float *dev_out)
{
    const double nn = sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
    if (!(fabs(nn - 1.0) < 1e-9)) {
        snprintf(m->err, sizeof(m->err), "loc_spectra_map: direction is not a unit vector");
        return LOC_EINVAL;
    }
    const double d[3] = {dir[0] / nn, dir[1] / nn, dir[2] / nn};
    double north[3] = {0.0, 0.0, 1.0};
    if (fabs(d[2]) > 1.0 - 1e-9) {
        north[1] = 1.0;
        north[2] = 0.0;
    }
    const double nd = north[0] * d[0] + north[1] * d[1] + north[2] * d[2];
    double e2[3] = {north[0] - nd * d[0], north[1] - nd * d[1], north[2] - nd * d[2]};
    const double l2 = sqrt(e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2]);
    for (int a = 0; a < 3; a++) e2[a] /= l2;
    const double e1[3] = {e2[1] * d[2] - e2[2] * d[1], e2[2] * d[0] - e2[0] * d[2], e2[0] * d[1] - e2[1] * d[0]};
    Dir3 D;
    loc_fill_dir(m, dir, &D);
    const double upc = (double)LOC_H0 / m->root_cm;  // grid units per cm
    const double sl[2] = {D.T[0] ? 4294967296.0 / (double)D.T[0] : 0.0, D.T[1] ? 4294967296.0 / (double)D.T[1] : 0.0};
    // working-frame coordinates of a model-frame point x (cm): w_k = flip ? W_k - u x_a : u x_a; of a vector: sign only
    double wc[3], w1[3], w2[3];
    for (int k = 0; k < 3; k++) {
        const int a = D.ax[k];
        const double sg = D.flip[k] ? -1.0 : 1.0;
        wc[k] = D.flip[k] ? (double)D.W[k] - upc * centre_cm[a] : upc * centre_cm[a];
        w1[k] = sg * upc * pixel_cm * e1[a];
        w2[k] = sg * upc * pixel_cm * e2[a];
    }
    const double cx = 0.5 * (nx - 1), cy = 0.5 * (ny - 1);
    double o[2], ex[2], ey[2];
    for (int k = 0; k < 2; k++) {
        ex[k] = w1[k + 1] - sl[k] * w1[0];
        ey[k] = w2[k + 1] - sl[k] * w2[0];
        o[k] = (wc[k + 1] - sl[k] * wc[0]) - cx * ex[k] - cy * ey[k];
    }
    return launch_spectra3d(m, trans, dir, nx, ny, o, ex, ey, dev_out);
}

// ---- line-area map (Fig. 5c: W = integral of T_A over velocity) -------------------------------------------
// One warp per pixel: coalesced reads of the pixel's spectrum, butterfly sum, W = dv[km/s] * sum_c T_A(c).  HBM bound:
// 4 nch bytes read per pixel, 4 written.
__global__ void __launch_bounds__(256) k_line_area(const float *__restrict__ cube, long long npix, int nch, float dv_kms, float *__restrict__ w)
{
    const int lane = threadIdx.x & 31;
    const long long pix = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    if (pix >= npix) return;
    const float *sp = cube + pix * nch;
    float a = 0.f;
    for (int c = lane; c < nch; c += 32) a += __ldg(sp + c);
    for (int o = 16; o >= 1; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) w[pix] = a * dv_kms;
}

int loc_launch_line_area(loc_model *m, const float *dev_cube, long long npix, float *dev_w)
{
    if (npix == 0) return LOC_OK;
    const long long threads = npix * 32;
    k_line_area<<<(unsigned)((threads + 255) / 256), 256, 0, m->stream>>>(dev_cube, npix, m->nch, (float)(m->dv * 1e-5), dev_w);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    return LOC_OK;
}

// ---- shell spectra without a workspace (include/loc.h, loc_spectra_shells_static) -----------------------------------------
// k_spectra1d reads two pieces of scratch that normally sit in the model's workspace: the device copy of the shell radii
// and the packed (velocity, total line width) record of every shell.  Here both sit in one array that is part of the
// library image, so the call needs neither a loc_model nor a byte of memory from the caller beyond inputs and outputs.
//   bytes [0, 8 MAX)        double r_out[MAX]
//   bytes [8 MAX, 24 MAX)   float4 kin[MAX]     (v_r, 0, 0, sqrt(sigma^2 + k T / m))
// Each call writes the first nshell entries of both parts before the kernel reads them and reads nothing beyond, so what an
// earlier call (possibly with more shells) left behind is never seen and nothing has to be cleared.
static __device__ __align__(256) unsigned char g_shell_scratch[LOC_STATIC_MAX_SHELLS * (sizeof(double) + sizeof(float4))];

#define LOC_STATIC_MAX_DEVICES 64
// g_shell_scratch is a host-side handle in host code, not an address a kernel can use; the device address differs per GPU
// and is looked up once per device, with that device current, on the first call made there.
static void *g_shell_scratch_addr[LOC_STATIC_MAX_DEVICES];
static std::mutex g_shell_scratch_mu;

// same arithmetic as k_pack_kin (loc_api.cu), written into the static array, which device code may name directly
__global__ void k_pack_kin_static(int n, const float *vr, const float *sigma, const float *tkin, double kT_over_m_per_K)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 *kin = reinterpret_cast<float4 *>(g_shell_scratch + LOC_STATIC_MAX_SHELLS * sizeof(double));
    const double s = sigma[i];
    const double st = sqrt(s * s + kT_over_m_per_K * (double)tkin[i]);  // DESIGN R3
    kin[i] = make_float4(vr[i], 0.0f, 0.0f, (float)st);
}

static int static_fail(char *err, int err_len, int code, const char *fmt, ...)
{
    if (err && err_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, (size_t)err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

extern "C" int loc_spectra_shells_static(int nshell, const double *r_out, const float *dev_vrad, const float *dev_sigma,
                                         const float *dev_tkin, double mass_amu, const float *dev_pop_u, const float *dev_pop_l,
                                         double freq_hz, double einstein_A, double g_upper, double g_lower, int nchannel,
                                         double band_halfwidth_cm_s, double t_background_K, int nlos, const double *offsets_cm,
                                         float *dev_out, void *stream, char *err, int err_len)
{
    if (err && err_len > 0) err[0] = 0;
    if (nshell > LOC_STATIC_MAX_SHELLS)
        return static_fail(err, err_len, LOC_EINVAL, "loc_spectra_shells_static: %d shells exceed LOC_STATIC_MAX_SHELLS = %d (the built-in scratch array); use loc_create_model + loc_spectra with a workspace for larger models", nshell, LOC_STATIC_MAX_SHELLS);
    if (nshell < 1 || nlos < 0) return static_fail(err, err_len, LOC_EINVAL, "loc_spectra_shells_static: nshell must be >= 1 and nlos >= 0");
    if (nchannel < 1 || nchannel > 1024) return static_fail(err, err_len, LOC_EINVAL, "loc_spectra_shells_static: nchannel must be in [1,1024]");
    if (!r_out || !dev_vrad || !dev_sigma || !dev_tkin || !dev_pop_u || !dev_pop_l || (nlos > 0 && (!offsets_cm || !dev_out)))
        return static_fail(err, err_len, LOC_EINVAL, "loc_spectra_shells_static: NULL argument");
    if (!(band_halfwidth_cm_s > 0.0) || !(t_background_K >= 0.0) || !(freq_hz > 0.0) || !(einstein_A > 0.0) || !(g_upper > 0.0) || !(g_lower > 0.0) || !(mass_amu >= 0.0))
        return static_fail(err, err_len, LOC_EINVAL, "loc_spectra_shells_static: band, frequency, A and statistical weights must be > 0; T_bg and mass >= 0");
    double prev = 0.0;
    for (int k = 0; k < nshell; k++) {
        if (!(r_out[k] > prev)) return static_fail(err, err_len, LOC_EINVAL, "loc_spectra_shells_static: shell radii must be positive and strictly ascending");
        prev = r_out[k];
    }
    if (nlos == 0) return LOC_OK;

    // once per device: the device address of the scratch array
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(err, err_len, LOC_ECUDA, "loc_spectra_shells_static: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= LOC_STATIC_MAX_DEVICES) return static_fail(err, err_len, LOC_EINVAL, "loc_spectra_shells_static: device ordinal %d not supported (< %d)", dev, LOC_STATIC_MAX_DEVICES);
    unsigned char *base;
    {
        std::lock_guard<std::mutex> lock(g_shell_scratch_mu);
        if (!g_shell_scratch_addr[dev]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_shell_scratch);
            if (e != cudaSuccess || !p)
                return static_fail(err, err_len, LOC_ECUDA, "loc_spectra_shells_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
            g_shell_scratch_addr[dev] = p;
        }
        base = static_cast<unsigned char *>(g_shell_scratch_addr[dev]);
    }
    double *d_rout = reinterpret_cast<double *>(base);
    float4 *d_kin = reinterpret_cast<float4 *>(base + LOC_STATIC_MAX_SHELLS * sizeof(double));
    cudaStream_t st = (cudaStream_t)stream;

    // stream-ordered behind whatever the previous call on this stream still reads from the array
    e = cudaMemcpyAsync(d_rout, r_out, sizeof(double) * nshell, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return static_fail(err, err_len, LOC_ECUDA, "loc_spectra_shells_static: cudaMemcpyAsync(r_out): %s", cudaGetErrorString(e));
    const double ktm = (mass_amu > 0.0) ? LOC_KB / (mass_amu * LOC_AMU) : 0.0;
    k_pack_kin_static<<<(nshell + 255) / 256, 256, 0, st>>>(nshell, dev_vrad, dev_sigma, dev_tkin, ktm);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(err, err_len, LOC_ECUDA, "loc_spectra_shells_static: k_pack_kin_static: %s", cudaGetErrorString(e));

    // the parameter block of k_spectra1d, filled as spec_common() fills it from a loc_model (no hyperfine structure)
    const double dv = 2.0 * band_halfwidth_cm_s / nchannel;
    SpecCommon C;
    memset(&C, 0, sizeof(C));
    C.nch = nchannel;
    C.nchp = (nchannel + 3) & ~3;
    C.dv = (float)dv;
    C.xmin = 6.0f;
    C.tk_per_occ = (float)(LOC_HP * freq_hz / LOC_KB);
    C.bgocc = (t_background_K > 0.0) ? (float)(1.0 / expm1(LOC_HP * freq_hz / (LOC_KB * t_background_K))) : 0.0f;
    C.ck = LOC_CL * LOC_CL * LOC_CL * einstein_A / (8.0 * LOC_PI * freq_hz * freq_hz * freq_hz * dv);
    C.gratio = g_upper / g_lower;
    C.ncell = nshell;
    C.pop_u = dev_pop_u;
    C.pop_l = dev_pop_l;
    C.kin = d_kin;
    C.nc = 1;
    C.wgt[0] = 1.0f;
    const size_t smem = sizeof(float) * LOC_SPEC_WARPS * C.nchp;
    for (int b0 = 0; b0 < nlos; b0 += LOC_SPEC_BATCH1D) {
        Spec1D P;
        P.C = C;
        P.C.out = dev_out + (int64_t)b0 * nchannel;
        P.ns = nshell;
        P.nlos = std::min(nlos - b0, LOC_SPEC_BATCH1D);
        P.r_out = d_rout;
        for (int i = 0; i < LOC_SPEC_BATCH1D; i++) P.b[i] = (i < P.nlos) ? offsets_cm[b0 + i] : 0.0;
        k_spectra1d<<<(P.nlos + LOC_SPEC_WARPS - 1) / LOC_SPEC_WARPS, 32 * LOC_SPEC_WARPS, smem, st>>>(P);
        e = cudaGetLastError();
        if (e != cudaSuccess) return static_fail(err, err_len, LOC_ECUDA, "loc_spectra_shells_static: k_spectra1d: %s", cudaGetErrorString(e));
    }
    return LOC_OK;
}
