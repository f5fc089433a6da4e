// loc_sim3d.cu -- 3D radiative kernel: replays the precomputed step streams (loc_paths3d.cu) every ALI iteration and
// evaluates, per ray step and velocity channel, the Doppler-shifted profile, the optical depth, the photon
// transfer of Eq. 3 and the two per-cell sums (Eq. 2 first term; escape fraction of PAPER.md:81) for all traced
// transitions at once (the "all transitions in one pass" option the paper leaves open).
//
// Work decomposition (DESIGN 6.4).  A warp carries FOUR rays at a time, one per quarter-warp ("group" of 8 lanes); a lane
// owns 4 CONSECUTIVE channels of the ray's local profile window (8 lanes x 4 = 32 channels per pass), so that
//   * the photon spectrum of a ray lives in shared memory and is read / written with one 128-bit access per lane and
//     transition, conflict free for any window position (a quarter-warp is one shared-memory phase);
//   * the sums over a lane's 4 channels are free, and the cross-lane reduction is an 8-lane halving butterfly whose every
//     instruction serves 4 ray steps;
//   * all per-step scalar work (record decode, Doppler shift, window, per-transition coefficients) is done lane-parallel
//     for 8 records x 4 rays at once in a "prepare" phase, not redundantly by 32 lanes per step.
// The four groups stay in lock step: every round each group consumes exactly one stream record (tasks are padded to
// whole chunks of 8 records by the path builder); the rare spectrum operations (background, save, load) are executed
// by the whole warp for the group that needs them.
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>

#include "loc_internal.cuh"

#define LOC_GROUPS 4  // rays per warp
#define LOC_CHUNK 8   // records per group and prepare phase (= LOC_TASK_ALIGN)
#define LOC_PASS 40   // channels per pass: 8 lanes x (one aligned float4 + one scalar)

struct Sim3D {
    int nch, nchp, nsp, nslot;
    int slot0;  // first counter / coefficient slot handled by this launch (transitions may be split over launches)
    float dv, xmin, eps_tau, inv_ndir;
    const Dir3 *dirs;
    const unsigned char *task_dir;
    const long long *task_off;
    const uint2 *stream;
    long long ntask;
    const float4 *kin;
    const float2 *coef;
    float2 *cnt;
    uint32_t *visits, *pathz;
    unsigned long long *nsteps;
    unsigned int *queue;
    float *pool;
    Selection S;
};

// per-record scalars written by the prepare phase (32 bytes)
struct __align__(16) RecPrep {
    float cc;        // profile centre in channel units: v0 / dv + (nch - 1) / 2
    float ky;        // dv sqrt(log2(e) / 2) / sigma :  phi = 2^(lamp - ((c - cc) ky)^2)
    float lamp;      // log2(dv / (sigma sqrt(2 pi)))
    float w;         // a s / V_eff = dzeta / (h NDIR)
    unsigned cell;   // STEP: cell index; SAVE / LOAD: slot
    unsigned opdz;   // opcode | level | dzeta (stream word)
    int clo, chi;    // channel window of the step
};

// per (record, transition) coefficients (16 bytes): X_c = thin ? phi + c0 (B2 + c0 (B3 + c0 B4)) : 1 - 2^(c0 phi)
//   n' = n + X (c1 + alpha n);  SJ += scale sum n X;  ESC += scale sum X
struct __align__(16) TPrep {
    float c0, c1, alpha, scale;
};

#define LOC_XCLIP 4.0f       // the window may be clipped to one 32-channel pass only outside +-4 sigma
#define LOC_THIN_TAU 0.03f  // line-centre optical depth of a step below which the cubic series of (1-e^-t)/t is used

template <int NT>
__device__ __forceinline__ void prepare_record(const Sim3D &P, uint2 rec, float d0, float d1, float d2, float sf, RecPrep *rp, TPrep *tp,
                                               unsigned &thickmask)
{
    RecPrep r;
    r.cell = rec.x;
    r.opdz = rec.y;
    r.cc = 0.f;
    r.ky = 0.f;
    r.lamp = 0.f;
    r.w = 0.f;
    r.clo = 0;
    r.chi = -1;
    thickmask = 0;
    if ((rec.y >> 24) == LOC_OP_STEP) {
        const float4 k = __ldg(P.kin + rec.x);
        const float v0 = -(k.x * d0 + k.y * d1 + k.z * d2);  // DESIGN R6
        const float sig = k.w;
        const unsigned dz = rec.y & 0x1fffffu;
        const int lev = (rec.y >> 21) & 7;
        const float s = (float)dz * sf;
        const float w = (float)dz * P.inv_ndir * __int_as_float((127 - LOC_LB + lev) << 23);
        const float inv_sig = __fdividef(1.0f, sig);
        const float amp = P.dv * 0.3989422804f * inv_sig;
        const float2 *cf = P.coef + (long long)rec.x * P.nsp + P.slot0;
        float tau0m = 0.f;
#pragma unroll
        for (int t = 0; t < NT; t++) {
            const float2 ke = __ldg(cf + t);
            const float ks = ke.x * s;
            const float tau0 = fabsf(ks) * amp;
            tau0m = fmaxf(tau0m, tau0);
            TPrep q;
            if (tau0 >= LOC_THIN_TAU) {
                thickmask |= 1u << t;
                q.c0 = -ks * LOC_LOG2E;
                q.c1 = __fdividef(ke.y, ke.x);  // source function in occupation-number units
                q.alpha = -1.0f;
                q.scale = __fdividef(w, ks);
            } else {
                q.c0 = ks;
                q.c1 = ke.y * s;
                q.alpha = -ks;
                q.scale = w;
            }
            tp[t] = q;
        }
        // window half-width in sigma: the profile mass left outside stays a fixed fraction (that of xmin at tau0 <= 1) of
        // the escape sum  sum_c phi_c f(tau_c) ~ 1/tau0  of an optically thick step (DESIGN 5.3)
        float X = P.xmin;
        if (tau0m > 1.0f) X = sqrtf(fmaf(2.0f, __logf(tau0m), X * X));
        const float inv_dv = __fdividef(1.0f, P.dv);
        r.cc = fmaf(v0, inv_dv, 0.5f * (float)(P.nch - 1));
        const float hw = X * sig * inv_dv;
        int clo = max(0, (int)ceilf(r.cc - hw)), chi = min(P.nch - 1, (int)floorf(r.cc + hw));
        // One pass of the kernel covers LOC_PASS = 40 channels starting at a multiple of 4.  If the window overshoots that by a few
        // channels, drop the outermost ones (never closer than LOC_XCLIP sigma to the line centre) instead of paying a
        // second pass; their profile mass is booked as escaping like everything outside the window (DESIGN 5.3).
        {
            const float lim = LOC_XCLIP * sig * inv_dv;
            int lo = clo, hi = chi;
#pragma unroll
            for (int i = 0; i < 3; i++) {
                if ((lo & 3) + (hi - lo + 1) <= LOC_PASS) break;
                if (r.cc - (float)lo > (float)hi - r.cc) lo++;
                else hi--;
            }
            if ((lo & 3) + (hi - lo + 1) <= LOC_PASS && r.cc - (float)lo >= lim && (float)hi - r.cc >= lim) {
                clo = lo;
                chi = hi;
            }
        }
        r.clo = clo;
        r.chi = chi;
        r.ky = P.dv * 0.8493218f * inv_sig;
        r.lamp = __log2f(amp);
        r.w = w;
    }
    *rp = r;
}

template <int NT, bool GEOM>
__global__ void __launch_bounds__(32) k_sim3d(Sim3D P)
{
    constexpr int NV = 2 * NT;                 // reduced values per step: a[t], b[t]
    constexpr int NPASS = (NV + 7) / 8;        // 8-lane butterflies of up to 8 values
    extern __shared__ __align__(16) float smem[];
    const int lane = threadIdx.x, grp = lane >> 3, l8 = lane & 7;
    const int nchp = P.nchp;
    const int spec = NT * nchp;                // floats per ray spectrum
    float *sn_all = smem;                                  // [4][NT][nchp]
    __shared__ TPrep tp_all[LOC_GROUPS * LOC_CHUNK * NT];    // [4][8][NT]   (separate objects: no aliasing with the spectra)
    __shared__ RecPrep rp_all[LOC_GROUPS * LOC_CHUNK];       // [4][8]
    float *sn = sn_all + grp * spec;
    TPrep *tpg = tp_all + grp * LOC_CHUNK * NT;
    RecPrep *rpg = rp_all + grp * LOC_CHUNK;
    float *slots_warp = P.pool + (long long)blockIdx.x * LOC_GROUPS * P.nslot * spec;

    long long off = 0, end = 0;  // this group's position in the stream
    bool done = false;
    float d0 = 0.f, d1 = 0.f, d2 = 0.f, sf = 0.f;
    unsigned long long mysteps = 0, myactive = 0;

    for (;;) {
        // ---- refill: groups whose task is exhausted take the next root ray from the queue ----
        {
            const bool need = !done && off >= end;
            long long task = 0;
            if (need && l8 == 0) task = atomicAdd(P.queue, 1u);
            task = __shfl_sync(0xffffffffu, task, grp * 8);
            if (need) {
                if (task >= P.ntask) {
                    done = true;
                } else {
                    const Dir3 *Dp = P.dirs + P.task_dir[task];
                    d0 = __ldg(&Dp->d[0]);
                    d1 = __ldg(&Dp->d[1]);
                    d2 = __ldg(&Dp->d[2]);
                    sf = __ldg(&Dp->sf);
                    off = __ldg(P.task_off + task);
                    end = __ldg(P.task_off + task + 1);
                }
            }
        }
        __syncwarp();
        if (__all_sync(0xffffffffu, done)) break;
        // ---- prepare: lane l8 of each group decodes record off + l8 of its ray ----
        uint2 rec = make_uint2(0u, LOC_OP_NOP << 24);
        if (!done && off + l8 < end) rec = __ldg(P.stream + off + l8);
        unsigned thick_l;
        prepare_record<NT>(P, rec, d0, d1, d2, sf, rpg + l8, tpg + l8 * NT, thick_l);
        off += LOC_CHUNK;
        __syncwarp();

        // ---- 8 rounds: every group consumes one record per round ----
        for (int r = 0; r < LOC_CHUNK; r++) {
            const RecPrep rp = rpg[r];
            const unsigned op = rp.opdz >> 24;
            const unsigned thick = __shfl_sync(0xffffffffu, thick_l, grp * 8 + r);
            // spectrum operations, executed by the whole warp for one group at a time
            unsigned ctrl = __ballot_sync(0xffffffffu, op == LOC_OP_BG || op == LOC_OP_SAVE || op == LOC_OP_LOAD) & 0x01010101u;
            while (ctrl) {
                const int g = (__ffs(ctrl) - 1) >> 3;
                ctrl &= ctrl - 1;
                const unsigned gop = __shfl_sync(0xffffffffu, op, g * 8), gx = __shfl_sync(0xffffffffu, rp.cell, g * 8);
                float *gs = sn_all + g * spec;
                float *slot = slots_warp + ((long long)g * P.nslot + gx) * spec;
                if (gop == LOC_OP_BG) {
#pragma unroll
                    for (int t = 0; t < NT; t++) {
                        const float b = P.S.bgocc[P.slot0 + t];
                        for (int c = lane; c < nchp; c += 32) gs[t * nchp + c] = b;
                    }
                } else if (gop == LOC_OP_SAVE) {
                    for (int i = lane * 4; i < spec; i += 128) *reinterpret_cast<float4 *>(slot + i) = *reinterpret_cast<const float4 *>(gs + i);
                } else {
                    for (int i = lane * 4; i < spec; i += 128) *reinterpret_cast<float4 *>(gs + i) = *reinterpret_cast<const float4 *>(slot + i);
                }
                __syncwarp();
            }
            const bool step = op == LOC_OP_STEP;
            const unsigned anystep = __ballot_sync(0xffffffffu, step);
            if (!anystep) continue;
            const unsigned any_thick = __reduce_or_sync(0xffffffffu, step ? thick : 0u);
            const unsigned any_thin = __reduce_or_sync(0xffffffffu, step ? ~thick : 0u);

            float a[NT], b[NT];
#pragma unroll
            for (int t = 0; t < NT; t++) a[t] = b[t] = 0.f;
            float sphi = 0.f;
            const TPrep *tpr = tpg + r * NT;
            // passes of 40 channels over the window (one pass unless the line is very thick): lane l8 owns the aligned
            // float4 at wb + 4 l8 and the single channel wb + 32 + l8
            int wb = rp.clo & ~3;
            const int chi = step ? rp.chi : -1;
            while (__any_sync(0xffffffffu, wb <= chi)) {
                const int cb = wb + 4 * l8, ce = wb + 32 + l8;
                float phi[5], B2[5], B3[5], B4[5];
#pragma unroll
                for (int k = 0; k < 5; k++) {
                    const int c = (k < 4) ? cb + k : ce;
                    const float y = ((float)c - rp.cc) * rp.ky;
                    const float e = ex2f(fmaf(-y, y, rp.lamp));
                    phi[k] = (c >= rp.clo && c <= chi) ? e : 0.0f;
                    sphi += phi[k];
                    const float p2 = phi[k] * phi[k];
                    B2[k] = -0.5f * p2;
                    B3[k] = (1.0f / 6.0f) * p2 * phi[k];
                    B4[k] = (-1.0f / 24.0f) * p2 * p2;
                }
                const bool inb = cb <= chi;            // chi < nch <= nchp and cb is a multiple of 4: the float4 is in range
                const bool ine = ce <= chi;
                float nn[NT][5];
#pragma unroll
                for (int t = 0; t < NT; t++) {
                    float4 n4 = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (inb) n4 = *reinterpret_cast<const float4 *>(sn + t * nchp + cb);
                    nn[t][0] = n4.x;
                    nn[t][1] = n4.y;
                    nn[t][2] = n4.z;
                    nn[t][3] = n4.w;
                    nn[t][4] = ine ? sn[t * nchp + ce] : 0.f;
                }
#pragma unroll
                for (int t = 0; t < NT; t++) {
                    const TPrep q = tpr[t];
                    const bool tk = (thick >> t) & 1u;
                    if (!((any_thick >> t) & 1u)) {  // every ray of the warp is thin in this transition
#pragma unroll
                        for (int k = 0; k < 5; k++) {
                            const float X = fmaf(q.c0, fmaf(q.c0, fmaf(q.c0, B4[k], B3[k]), B2[k]), phi[k]);
                            a[t] = fmaf(nn[t][k], X, a[t]);
                            b[t] += X;
                            nn[t][k] = fmaf(X, fmaf(q.alpha, nn[t][k], q.c1), nn[t][k]);
                        }
                    } else if (!((any_thin >> t) & 1u)) {  // every ray is thick
#pragma unroll
                        for (int k = 0; k < 5; k++) {
                            const float X = 1.0f - ex2f(q.c0 * phi[k]);
                            a[t] = fmaf(nn[t][k], X, a[t]);
                            b[t] += X;
                            nn[t][k] = fmaf(X, fmaf(q.alpha, nn[t][k], q.c1), nn[t][k]);
                        }
                    } else {  // mixed: both forms, selected per ray
#pragma unroll
                        for (int k = 0; k < 5; k++) {
                            const float Xs = fmaf(q.c0, fmaf(q.c0, fmaf(q.c0, B4[k], B3[k]), B2[k]), phi[k]);
                            const float Xe = 1.0f - ex2f(q.c0 * phi[k]);
                            const float X = tk ? Xe : Xs;
                            a[t] = fmaf(nn[t][k], X, a[t]);
                            b[t] += X;
                            nn[t][k] = fmaf(X, fmaf(q.alpha, nn[t][k], q.c1), nn[t][k]);
                        }
                    }
                }
#pragma unroll
                for (int t = 0; t < NT; t++) {
                    if (inb) *reinterpret_cast<float4 *>(sn + t * nchp + cb) = make_float4(nn[t][0], nn[t][1], nn[t][2], nn[t][3]);
                    if (ine) sn[t * nchp + ce] = nn[t][4];
                }
                wb += LOC_PASS;
            }
            // ---- reductions over the 8 lanes of each group ----
            sphi += __shfl_xor_sync(0xffffffffu, sphi, 4);
            sphi += __shfl_xor_sync(0xffffffffu, sphi, 2);
            sphi += __shfl_xor_sync(0xffffffffu, sphi, 1);
            float v[NPASS * 8];
#pragma unroll
            for (int i = 0; i < NPASS * 8; i++) v[i] = 0.f;
#pragma unroll
            for (int t = 0; t < NT; t++) {
                v[t] = a[t];
                v[NT + t] = b[t];
            }
            float tot[NPASS];
#pragma unroll
            for (int p = 0; p < NPASS; p++) {
                float *u = v + 8 * p;
                {
                    const bool up = l8 & 4;
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        const float keep = up ? u[i + 4] : u[i], send = up ? u[i] : u[i + 4];
                        u[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
                    }
                }
                {
                    const bool up = l8 & 2;
#pragma unroll
                    for (int i = 0; i < 2; i++) {
                        const float keep = up ? u[i + 2] : u[i], send = up ? u[i] : u[i + 2];
                        u[i] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
                    }
                }
                {
                    const bool up = l8 & 1;
                    const float keep = up ? u[1] : u[0], send = up ? u[0] : u[1];
                    tot[p] = keep + __shfl_xor_sync(0xffffffffu, send, 1);
                }
            }
            // lane l8 of a group now holds the group totals of values 4*bit2 + 2*bit1 + bit0 ... = l8, 8 + l8, 16 + l8
            if (step) {
                float2 *cn = P.cnt + (long long)rp.cell * P.nsp + P.slot0;
                const float wesc = rp.w - rp.w * sphi;  // photons emitted outside the window escape (DESIGN 5.3)
#pragma unroll
                for (int p = 0; p < NPASS; p++) {
                    const int i = 8 * p + l8;
                    if (i < NT)
                        atomicAdd(&cn[i].x, tot[p] * tpr[i].scale);
                    else if (i < NV)
                        atomicAdd(&cn[i - NT].y, fmaf(tot[p], tpr[i - NT].scale, wesc));
                }
                if (l8 == 0) {
                    mysteps++;
                    if (GEOM) {
                        atomicAdd(&P.visits[rp.cell], 1u);
                        atomicAdd(&P.pathz[rp.cell], rp.opdz & 0x1fffffu);
                        const float h5 = 5.0f * 0.8493218f / rp.ky;  // 5 sigma in channels
                        myactive += max(0, min(P.nch - 1, (int)floorf(rp.cc + h5)) - max(0, (int)ceilf(rp.cc - h5)) + 1);
                    }
                }
            }
            __syncwarp();
        }
    }
    // per-warp totals
    for (int o = 16; o >= 1; o >>= 1) {
        mysteps += __shfl_xor_sync(0xffffffffu, mysteps, o);
        myactive += __shfl_xor_sync(0xffffffffu, myactive, o);
    }
    if (lane == 0 && mysteps) atomicAdd(P.nsteps, mysteps);
    if (GEOM && lane == 0 && myactive) atomicAdd(P.nsteps + 1, myactive);
}

template <int NT>
static int launch3d(loc_model *m, Sim3D &P, int geom)
{
    const size_t smem = sizeof(float) * LOC_GROUPS * NT * P.nchp;  // + static: TPrep / RecPrep tables
    if (smem > 220 * 1024) {
        snprintf(m->err, sizeof(m->err), "nchannel * ntrans too large for the shared-memory spectra (%zu bytes per warp)", smem);
        return LOC_EINVAL;
    }
    auto kern = geom ? k_sim3d<NT, true> : k_sim3d<NT, false>;
    LOC_CUDA_CHECK(m, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int bps = 0;
    LOC_CUDA_CHECK(m, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, 32, smem));
    if (bps < 1) bps = 1;
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, 0);
    long long blocks = (long long)nsm * bps;
    blocks = std::min<long long>(blocks, (m->ntask + LOC_GROUPS - 1) / LOC_GROUPS);
    blocks = std::min<long long>(blocks, m->max_warps);
    if (blocks < 1) blocks = 1;
    LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_queue, 0, sizeof(unsigned int), m->stream));
    kern<<<(unsigned)blocks, 32, smem, m->stream>>>(P);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    return LOC_OK;
}

int loc_launch_sim3d(loc_model *m, int geom)
{
    Sim3D P;
    P.nch = m->nch;
    P.nchp = (m->nch + 3) & ~3;
    P.nsp = m->selh.nsp;
    P.nslot = std::max(m->nlev - 1, 1);
    P.dv = (float)m->dv;
    P.xmin = m->xmin;
    P.eps_tau = m->eps_tau;
    P.inv_ndir = 1.0f / (float)m->ndir;
    P.dirs = m->d_dirs;
    P.task_dir = m->d_task_dir;
    P.task_off = m->d_task_off;
    P.stream = m->d_stream;
    P.ntask = m->ntask;
    P.kin = m->kin;
    P.coef = m->coef;
    P.cnt = m->cnt;
    P.visits = m->visits;
    P.pathz = m->pathz;
    P.nsteps = m->d_steps;
    P.queue = m->d_queue;
    P.pool = m->spec_pool;
    P.S = m->selh;
    // Transitions are traced in `npart` launches of nearly equal size: the per-ray spectra of one launch then need less
    // shared memory, so more rays are in flight per SM (latency hiding), at the price of repeating the per-step scalar
    // work once per launch.  Default: parts of at most 5 transitions.
    int nsel = m->selh.nsel;
    int npart = (nsel + 4) / 5;
    if (getenv("LOC_SIM3D_PARTS")) npart = std::max(1, std::min(nsel, atoi(getenv("LOC_SIM3D_PARTS"))));
    int slot = 0;
    for (int part = 0; part < npart; part++) {
        int n = (nsel - slot + (npart - part) - 1) / (npart - part);
        P.slot0 = slot;
        int rc = LOC_EINVAL;
        // the step / active-channel statistics are taken by the first part only
        int g = geom && part == 0;
        unsigned long long *keep = P.nsteps;
        if (part > 0) P.nsteps = m->d_steps + 2;  // scratch slot
        switch (n) {
#define C3(N)                        \
    case N:                          \
        rc = launch3d<N>(m, P, g);   \
        break;
            C3(1) C3(2) C3(3) C3(4) C3(5) C3(6) C3(7) C3(8) C3(9) C3(10) C3(11) C3(12)
#undef C3
        }
        P.nsteps = keep;
        if (rc != LOC_OK) return rc;
        slot += n;
    }
    return LOC_OK;
}
