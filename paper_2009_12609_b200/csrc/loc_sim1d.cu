// loc_sim1d.cu -- 1D shell-ray simulation kernel (Eqs. 1-3).
//
// One WARP per ray (impact parameter); the spherical symmetry makes the ray a fixed sequence of shells (in through
// NS-1..k0, out through k0+1..NS-1) with precomputed path lengths.  See k_sim1d_w below.  The paper's kernel
// used one work item per ray and one transition at a time.  (Round 1 also had a
// block-per-ray kernel with one thread per channel; it was 2.9x slower on C2 and unreachable for every legal input, and
// was removed: profiles/r1_sim1d_C2.md keeps its measurements.)
#include <stdio.h>
#include <stdlib.h>

#include "loc_internal.cuh"

struct Sim1D {
    int ns, nch, nsp;
    float dv, xmin, eps_tau;
    const int *order, *k0;
    const long long *off;
    const float *tabs, *tabmu, *tabw;
    const float4 *kin;
    const float2 *coef;
    float2 *cnt;
    uint32_t *visits;
    unsigned long long *nactive;
    Selection S;
    HfsTab H;
};

__device__ __forceinline__ void seg1d(const Sim1D &P, int j, int nin, int k0, long long off, int &k, float &s, float &mu, float &w)
{
    if (j < nin) {  // inbound through shell NS-1-j
        k = P.ns - 1 - j;
        s = __ldg(P.tabs + off + (k - k0));
        w = __ldg(P.tabw + off + (k - k0));
        mu = -__ldg(P.tabmu + off + (k - k0));
    } else if (j == nin) {  // tangent shell, one step (DESIGN R5)
        k = k0;
        s = __ldg(P.tabs + off);
        w = __ldg(P.tabw + off);
        mu = -__ldg(P.tabmu + off);
    } else {  // outbound: entry cosine is that of the inner boundary r_{k-1}
        k = k0 + (j - nin);
        s = __ldg(P.tabs + off + (k - k0));
        w = __ldg(P.tabw + off + (k - k0));
        mu = __ldg(P.tabmu + off + (k - 1 - k0));
    }
}

// ------------------------------------------------------------------------------------------------------------------
// k_sim1d_w: one WARP per ray (profiles/r1_sim1d_C2.md: a block-per-ray kernel was issue bound at 2600 warp
// instructions per ray step, most of them per-step scalar work repeated by every warp of the block and a two-stage
// reduction).  The ray's spectra [NT][nchp] live in shared memory; per step the lanes cover the profile window in
// aligned quads of channels (one 128-bit shared-memory access per lane and transition, conflict free), sum their
// channels in registers, and ONE halving-butterfly reduction per step leaves each of the 2 NT + 1 totals in one lane,
// which issues the counter's atomic itself: no block barrier, no second reduction stage.  The step's table entries, cell
// kinematics and line coefficients are loaded one step ahead.
// ------------------------------------------------------------------------------------------------------------------
#define LOC_1D_WARPS 1  // rays per block (C2: 1 -> 3.80 ms, 2 -> 4.15 ms, 4 -> 4.13 ms: 24 instead of 22 resident rays per SM, finer scheduling)

struct Step1D {
    int k;
    float s, mu, w;
    float4 kin;
    float2 ke;  // lanes < NT: (kap, em) of transition `lane`
};

template <int NT>
__device__ __forceinline__ void load_step1d(const Sim1D &P, int j, int nin, int k0, long long off, int lane, Step1D &S)
{
    seg1d(P, j, nin, k0, off, S.k, S.s, S.mu, S.w);
    S.kin = __ldg(P.kin + S.k);
    if (lane < NT) S.ke = __ldg(P.coef + (long long)S.k * P.nsp + lane);
}

// HFS: some traced transition has hyperfine structure (loc_set_hyperfine): every transition then gets its own profile, the
// sum over its components, evaluated over ONE window that covers the components of all transitions; the sum of the sampled
// profile is folded into the escape sum transition by transition (b_t -= g_t sum phi_t), and with GEOM the active channels
// are counted per transition (within 5 sigma of any of its components).
template <int NT, bool GEOM, bool HFS>
__global__ void __launch_bounds__(LOC_1D_WARPS * 32) k_sim1d_w(Sim1D P, int nray)
{
    constexpr int NV = HFS ? 2 * NT : 2 * NT + 1;
    extern __shared__ __align__(16) float s_w[];  // per warp: [NT][nchp] spectra, then NT TParam
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int slot = blockIdx.x * LOC_1D_WARPS + warp;
    if (slot >= nray) return;  // the warps of a block never synchronise with each other
    const int nchp = (P.nch + 3) & ~3;
    float *sn = s_w + warp * (NT * nchp + 4 * NT);
    TParam *stp = reinterpret_cast<TParam *>(sn + NT * nchp);
    const int ray = P.order[slot];
    const int k0 = P.k0[ray];
    const long long off = P.off[ray];
    const int nin = P.ns - 1 - k0, nseg = 2 * nin + 1;
#pragma unroll
    for (int t = 0; t < NT; t++) {
        const float bg = P.S.bgocc[t];  // Eq. 1: background photons, as occupation number
        for (int c = lane; c < nchp; c += 32) sn[t * nchp + c] = bg;
    }
    const float inv_dv = 1.0f / P.dv, chalf = 0.5f * (float)(P.nch - 1);
    unsigned long long nact = 0;
    Step1D cur, nxt;
    cur.ke = nxt.ke = make_float2(0.f, 0.f);
    load_step1d<NT>(P, 0, nin, k0, off, lane, cur);

    for (int j = 0; j < nseg; j++) {
        nxt = cur;
        if (j + 1 < nseg) load_step1d<NT>(P, j + 1, nin, k0, off, lane, nxt);  // used one iteration later
        const float s = cur.s, w = cur.w, sig = cur.kin.w;
        const float v0 = -cur.kin.x * cur.mu;  // DESIGN R6, mu at the entry of the step
        const float amp = P.dv * 0.3989422804f / sig;
        __syncwarp();  // the previous step's reads of stp and writes of the spectra are done
        float tau0 = 0.f;
        if (lane < NT) {
            stp[lane] = make_tparam(cur.ke, s, w, amp);
            tau0 = fabsf(cur.ke.x * s) * amp;
        }
        const float tau0m = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(tau0)));
        __syncwarp();
        // ---- profile window of this step (DESIGN 5.3) ----
        // channels wider than the line (dv > sigma): the neglected sampled values are amp e^{-X^2/2} with amp ~ dv/sigma > 1,
        // and the sum of the sampled profile may be well below 1, so the window grows by 2 ln (dv/sigma)^2 (DESIGN 5.3)
        const float und = P.dv / sig;
        float X = P.xmin;
        if (und > 1.0f) X = sqrtf(fmaf(4.0f, __logf(und), X * X));
        if (tau0m > P.eps_tau) X = fmaxf(X, sqrtf(2.0f * __logf(tau0m / P.eps_tau)));
        const float cc = v0 * inv_dv + chalf;
        const float hw = X * sig * inv_dv;
        const int c_lo = max(0, (int)ceilf(cc + (HFS ? P.H.lo : 0.0f) - hw)), c_hi = min(P.nch - 1, (int)floorf(cc + (HFS ? P.H.hi : 0.0f) + hw));
        if (GEOM && !HFS) {
            const float h5 = 5.0f * sig * inv_dv;
            nact += (unsigned long long)max(0, min(P.nch - 1, (int)floorf(cc + h5)) - max(0, (int)ceilf(cc - h5)) + 1);
        }
        const float ky = 0.8493218f / sig;  // sqrt(log2(e)/2) / sigma
        const float lamp = __log2f(amp);
        float v[NV];
#pragma unroll
        for (int i = 0; i < NV; i++) v[i] = 0.f;
        if (HFS) {
            const float kyc = ky * P.dv;  // per channel
            for (int cb = (c_lo & ~3) + 4 * lane; cb <= c_hi; cb += 128) {
#pragma unroll
                for (int t = 0; t < NT; t++) {
                    float phi[4] = {0.f, 0.f, 0.f, 0.f};
                    bool act[4] = {false, false, false, false};
                    for (int q = 0; q < P.H.nc[t]; q++) {
                        const float wq = P.H.w[t][q], dq = P.H.dch[t][q];
#pragma unroll
                        for (int i = 0; i < 4; i++) {
                            const int c = cb + i;
                            const float y = ((float)c - cc - dq) * kyc;
                            const bool in = c >= c_lo && c <= c_hi;
                            phi[i] = in ? fmaf(wq, ex2f(fmaf(-y, y, lamp)), phi[i]) : phi[i];
                            act[i] |= in && y * y <= 18.033688f;  // |v - v0 - dv_q| <= 5 sigma
                        }
                    }
                    if (GEOM) nact += (unsigned long long)((int)act[0] + (int)act[1] + (int)act[2] + (int)act[3]);
                    const TParam tp = stp[t];
                    float4 n4 = *reinterpret_cast<float4 *>(sn + t * nchp + cb);
                    f32x2 n01 = pk2(n4.x, n4.y), n23 = pk2(n4.z, n4.w);
                    channel_update4(n01, n23, pk2(phi[0], phi[1]), pk2(phi[2], phi[3]), tp, v[t], v[NT + t]);
                    // photons emitted outside the window escape: w (1 - sum phi_t), as -g_t sum phi_t in the units of b_t
                    v[NT + t] = fmaf(tp.thick ? tp.c0 * (1.0f / LOC_LOG2E) : -1.0f, (phi[0] + phi[1]) + (phi[2] + phi[3]), v[NT + t]);
                    upk2(n01, n4.x, n4.y);
                    upk2(n23, n4.z, n4.w);
                    *reinterpret_cast<float4 *>(sn + t * nchp + cb) = n4;
                }
            }
        } else
        for (int cb = (c_lo & ~3) + 4 * lane; cb <= c_hi; cb += 128) {
            float phi[4];
#pragma unroll
            for (int i = 0; i < 4; i++) {
                const int c = cb + i;
                const float y = (((float)c - chalf) * P.dv - v0) * ky;
                phi[i] = (c >= c_lo && c <= c_hi) ? ex2f(fmaf(-y, y, lamp)) : 0.0f;
            }
            v[2 * NT] += (phi[0] + phi[1]) + (phi[2] + phi[3]);
            const f32x2 phi01 = pk2(phi[0], phi[1]), phi23 = pk2(phi[2], phi[3]);
#pragma unroll
            for (int t = 0; t < NT; t++) {
                const TParam tp = stp[t];
                float4 n4 = *reinterpret_cast<float4 *>(sn + t * nchp + cb);
                f32x2 n01 = pk2(n4.x, n4.y), n23 = pk2(n4.z, n4.w);
                channel_update4(n01, n23, phi01, phi23, tp, v[t], v[NT + t]);
                upk2(n01, n4.x, n4.y);
                upk2(n23, n4.z, n4.w);
                *reinterpret_cast<float4 *>(sn + t * nchp + cb) = n4;
            }
        }
        int owner;
        const float tot = warp_multi_reduce<NV>(v, lane, owner);
        float sphi = 0.0f;  // (HFS: already folded into the escape sums)
        if (!HFS) {
            const unsigned mphi = __ballot_sync(0xffffffffu, owner == 2 * NT);
            sphi = __shfl_sync(0xffffffffu, tot, __ffs(mphi) - 1);
        }
        if (owner >= 0 && owner < 2 * NT) {
            const int t = owner < NT ? owner : owner - NT;
            float2 *cn = P.cnt + (long long)cur.k * P.nsp + t;
            float val = tot * stp[t].scale;
            // photons emitted outside the window escape (DESIGN 5.3): w (1 - sum phi)
            if (owner >= NT) val += fmaf(-w, sphi, w);
            atomicAdd(owner < NT ? &cn->x : &cn->y, val);
        }
        if (GEOM && lane == 0) atomicAdd(&P.visits[cur.k], 1u);
        cur = nxt;
    }
    if (GEOM) {  // active updates of the ray, summed over the traced transitions (loc_stats.active_updates)
        if (HFS) {
            for (int o = 16; o >= 1; o >>= 1) nact += __shfl_xor_sync(0xffffffffu, nact, o);
        } else {
            nact *= NT;
        }
        if (lane == 0 && nact) atomicAdd(P.nactive, nact);
    }
}

template <int NT>
static int launch1d(loc_model *m, const Sim1D &P, int geom)
{
    // the spectra of a ray ([NT][nchp] floats, <= 12 x 1024 x 4 B = 48 KB for every legal input) live in shared memory
    const int nchp = (m->nch + 3) & ~3;
    const size_t smem_w = sizeof(float) * LOC_1D_WARPS * ((size_t)NT * nchp + 4 * NT);
    if (smem_w > 200 * 1024) {
        snprintf(m->err, sizeof(m->err), "nchannel * ntrans too large for the shared-memory spectra of the 1D kernel (%zu bytes)", smem_w);
        return LOC_EINVAL;
    }
    const int blocks = (m->nray + LOC_1D_WARPS - 1) / LOC_1D_WARPS;
#define LOC_L1(G, HF)                                                                                                             \
    do {                                                                                                                          \
        LOC_CUDA_CHECK(m, cudaFuncSetAttribute(k_sim1d_w<NT, G, HF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_w)); \
        k_sim1d_w<NT, G, HF><<<blocks, LOC_1D_WARPS * 32, smem_w, m->stream>>>(P, m->nray);                                    \
    } while (0)
    if (P.H.any) {
        if (geom) LOC_L1(true, true);
        else LOC_L1(false, true);
    } else {
        if (geom) LOC_L1(true, false);
        else LOC_L1(false, false);
    }
#undef LOC_L1
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    return LOC_OK;
}

int loc_launch_sim1d(loc_model *m, int geom)
{
    Sim1D P;
    P.ns = m->nshell;
    P.nch = m->nch;
    P.nsp = m->selh.nsp;
    P.dv = (float)m->dv;
    P.xmin = m->xmin;
    P.eps_tau = m->eps_tau;
    P.order = m->d_order;
    P.k0 = m->d_k0;
    P.off = m->d_off;
    P.tabw = m->d_tabw;
    P.tabs = m->d_tabs;
    P.tabmu = m->d_tabmu;
    P.kin = m->kin;
    P.coef = m->coef;
    P.cnt = m->cnt;
    P.visits = m->visits;
    P.nactive = m->d_steps + 1;
    P.S = m->selh;
    loc_fill_hfs(m, P.H);
    switch (m->selh.nsel) {
#define C1(N) \
    case N:   \
        return launch1d<N>(m, P, geom);
        C1(1) C1(2) C1(3) C1(4) C1(5) C1(6) C1(7) C1(8) C1(9) C1(10) C1(11) C1(12)
#undef C1
    }
    snprintf(m->err, sizeof(m->err), "unsupported number of traced transitions %d", m->selh.nsel);
    return LOC_EINVAL;
}
