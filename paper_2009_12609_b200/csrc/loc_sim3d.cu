// loc_sim3d.cu -- 3D radiative kernel: replays the precomputed step streams (loc_paths3d.cu) every ALI iteration and
// evaluates, per ray step and velocity channel, the Doppler-shifted profile, the optical depth, the photon
// transfer of Eq. 3 and the two per-cell sums (Eq. 2 first term; escape fraction of PAPER.md:81) for all traced
// transitions at once (the "all transitions in one pass" option the paper leaves open).
//
// Work decomposition (DESIGN 6.4).  A warp carries FOUR rays at a time, one per quarter-warp ("group" of 8 lanes).  Every
// step touches a SPAN of 32 consecutive channels that starts at a multiple of 4 and is centred on the Doppler-shifted
// line; lane l8 of the group owns the aligned quad  span + 4 l8 .. + 3, so that
//   * the photon spectrum of a ray lives in shared memory and is read / written with one 128-bit access per lane and
//     transition, conflict free for any span position (a quarter-warp is one shared-memory phase);
//   * the per-channel arithmetic is done on packed pairs (fma.rn.f32x2): the kernel is bound by instruction issue and by
//     the 16-lane ALU pipe (selects, compares, logic: 2 cycles each), not by FP32 throughput, so the common path has no
//     masks and no selects at all -- a span always lies inside the band, and channels of the span outside the nominal
//     window are simply updated too;
//   * the sums over a lane's 4 channels are free, and the cross-lane reduction is an 8-lane halving butterfly whose every
//     instruction serves 4 ray steps;
//   * all per-step scalar work (record decode, Doppler shift, window, per-transition coefficients, classification of the
//     round) is done lane-parallel for 8 records x 4 rays at once in a "prepare" phase.
// Steps whose window does not fit one span (very thick lines, bands narrower than 32 channels) take a masked multi-pass
// path.  The four groups stay in lock step: every round each group consumes exactly one stream record (tasks are padded
// to whole chunks of 8 records by the path builder); the rare spectrum operations (background, save, load) are executed
// by the whole warp for the group that needs them.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>

#include "loc_internal.cuh"

#define LOC_GROUPS 4  // rays per warp
#define LOC_CHUNK 8   // records per group and prepare phase (= LOC_TASK_ALIGN)
#define LOC_SPAN 32   // channels per pass: 8 lanes x one aligned float4

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

// Per-record scalars every lane of the group reads each round (16 bytes, one broadcast LDS.128).
//   y(channel wb + j) = A + j ky ;  phi = 2^(lamp - y^2)
// wbop: bits 0..9 first channel of the span, bits 10..21 per-transition "thick" flags, bit 31 = the record is a STEP
struct __align__(16) RecS {
    float A, ky, lamp;
    unsigned wbop;
};
#define LOC_WB_MASK 0x3ffu
#define LOC_THICK_SHIFT 10
#define LOC_RS_STEP 0x80000000u

// Class word of a round (one per chunk record index, OR over the four groups):
//   bits 0..11 some stepping ray MUST use the exponential form in transition t (tau0 > LOC_SER_TAU),
//   bits 12..23 some stepping ray MUST use the series (tau0 < LOC_EXP_TAU),
//   bit 24 a spectrum operation is due, bit 25 some group steps, bit 26 some stepping group needs the masked path
#define LOC_CLS_THIN_SHIFT 12
#define LOC_CLS_CTRL (1u << 24)
#define LOC_CLS_STEP (1u << 25)
#define LOC_CLS_SLOW (1u << 26)

#define LOC_XCLIP 3.9f     // a span may cut the nominal window, but never closer than this many sigma to the line centre
// Two forms of the per-channel factor (DESIGN 5.3).  Exponential: X = 1 - 2^(c0 phi), accurate (ex2.approx plus the
// subtraction) only while the line-centre optical depth of the step is >= LOC_EXP_TAU.  Series: X = phi f(tau) with
// f = 1 - tau/2 + tau^2/6 - tau^3/24 + tau^4/120, truncation < 2e-6 while tau0 <= LOC_SER_TAU.  In between either form
// will do, so a round whose four steps do not hold both extremes runs ONE form for the transition.
#define LOC_EXP_TAU 0.03f
#define LOC_SER_TAU 0.3f

// shared-memory tables of one warp, written by the prepare phase
template <int NT>
struct WarpTables {
    static constexpr int ROW = 10;                                  // float2 per row of partial sums (8 used): 80 bytes
    static constexpr int PGW = NT * ROW * 2;                        // words per group ...
    static constexpr int PG = (PGW + ((48 - PGW % 32) % 32)) / 2;   // ... padded to 16 mod 32 words (float2 units)
    RecS rs[LOC_GROUPS][LOC_CHUNK];
    float2 tp[LOC_GROUPS][LOC_CHUNK][NT];   // (c0, c1):  X_c = series ? phi + c0 (B2 + c0 (B3 + c0 (B4 + c0 B5))) : 1 - 2^(c0 phi)
                                            //            n' = n + X (c1 + alpha n),  alpha = series ? -c0 : -1
    unsigned cell[LOC_GROUPS][LOC_CHUNK];   // STEP: cell index; SAVE / LOAD: slot
    unsigned opdz[LOC_GROUPS][LOC_CHUNK];   // opcode | level | dzeta (stream word)
    float w[LOC_GROUPS][LOC_CHUNK];         // a s / V_eff = dzeta / (h NDIR)
    int2 win[LOC_GROUPS][LOC_CHUNK];        // nominal channel window [clo, chi] (masked path)
    unsigned cls[LOC_CHUNK];
    float2 part[LOC_GROUPS][PG];            // per-lane partial sums (a_t, b_t) of the round: [group][t][lane] (rows of 10)
};

// Prepare phase: lane (g, j) decodes record j of the chunk of group g, loads the cell's kinematics and line coefficients
// and fills the tables, including the class word of round j (the same for the four groups).
template <int NT>
__device__ __forceinline__ void prepare_record(const Sim3D &P, uint2 rec, float d0, float d1, float d2, float sf, WarpTables<NT> &T, int g,
                                               int j)
{
    RecS r;
    r.A = 0.f;
    r.ky = 0.f;
    r.lamp = -INFINITY;  // phi = 2^(-inf) = 0 for records that are not steps: the round leaves their spectra untouched
    r.wbop = 0u;
    T.cell[g][j] = rec.x;
    T.opdz[g][j] = rec.y;
    const unsigned op = rec.y >> 24;
    const bool step = op == LOC_OP_STEP;
    unsigned cls = (op == LOC_OP_BG || op == LOC_OP_SAVE || op == LOC_OP_LOAD) ? LOC_CLS_CTRL : 0u;
    float2 ke[NT];
    float s = 0.f, w = 0.f, amp = 0.f, tau0m = 0.f;
    float4 k = make_float4(0.f, 0.f, 0.f, 1.f);
    unsigned mexp = 0u, mser = 0u;
    if (step) {
        k = __ldg(P.kin + rec.x);
        const unsigned dz = rec.y & 0x1fffffu;
        const int lev = (rec.y >> 21) & 7;
        s = (float)dz * sf;
        w = (float)dz * P.inv_ndir * __int_as_float((127 - LOC_LB + lev) << 23);
        amp = P.dv * 0.3989422804f * __fdividef(1.0f, k.w);
        const float2 *cf = P.coef + (long long)rec.x * P.nsp + P.slot0;
#pragma unroll
        for (int t = 0; t < NT; t++) {
            ke[t] = __ldg(cf + t);
            const float tau0 = fabsf(ke[t].x * s) * amp;
            tau0m = fmaxf(tau0m, tau0);
            if (tau0 > LOC_SER_TAU) mexp |= 1u << t;
            if (tau0 < LOC_EXP_TAU) mser |= 1u << t;
        }
        cls |= LOC_CLS_STEP | mexp | (mser << LOC_CLS_THIN_SHIFT);
    } else {
#pragma unroll
        for (int t = 0; t < NT; t++) ke[t] = make_float2(0.f, 0.f);
    }
    unsigned thick = 0u;
    if (step) {
        // window half-width in sigma: the profile mass left outside stays a fixed fraction (that of xmin at tau0 <= 1) of
        // the escape sum  sum_c phi_c f(tau_c) ~ 1/tau0  of an optically thick step (DESIGN 5.3)
        const float v0 = -(k.x * d0 + k.y * d1 + k.z * d2);  // DESIGN R6
        float X = P.xmin;
        if (tau0m > 1.0f) X = sqrtf(fmaf(2.0f, __logf(tau0m), X * X));
        const float inv_dv = __fdividef(1.0f, P.dv);
        const float cc = fmaf(v0, inv_dv, 0.5f * (float)(P.nch - 1));
        const float sigch = k.w * inv_dv;
        const float hw = X * sigch;
        const int clo = max(0, (int)ceilf(cc - hw)), chi = min(P.nch - 1, (int)floorf(cc + hw));
        // the span: 32 channels from a multiple of 4, centred on the line, inside the band
        const int wbmax = (P.nch - LOC_SPAN) & ~3;
        int wb = 4 * (int)rintf((cc - 15.5f) * 0.25f);
        wb = max(0, min(wb, wbmax));
        const float lim = LOC_XCLIP * sigch;
        const bool fast = P.nch >= LOC_SPAN && (clo >= wb || cc - (float)wb >= lim) && (chi <= wb + LOC_SPAN - 1 || (float)(wb + LOC_SPAN - 1) - cc >= lim);
        if (P.nch < LOC_SPAN) wb = 0;
        if (!fast) {
            cls |= LOC_CLS_SLOW;
            T.win[g][j] = make_int2(clo, chi);
        }
        r.ky = 0.8493218f * __fdividef(1.0f, sigch);  // sqrt(log2(e) / 2) in channel units
        r.A = ((float)wb - cc) * r.ky;
        r.lamp = __log2f(amp);
        r.wbop = (unsigned)wb | LOC_RS_STEP;
    } else {
        T.win[g][j] = make_int2(0, -1);
    }
    T.w[g][j] = w;
    // class of the round: OR over the four groups (lanes j, 8 + j, 16 + j, 24 + j)
    cls |= __shfl_xor_sync(0xffffffffu, cls, 8);
    cls |= __shfl_xor_sync(0xffffffffu, cls, 16);
    if (g == 0) T.cls[j] = cls;
    const unsigned any_exp = cls & 0xfffu, any_ser = (cls >> LOC_CLS_THIN_SHIFT) & 0xfffu;
    // form per transition: the series unless some ray of the round must use the exponential; in a round that holds both
    // extremes every ray takes the form its own tau0 prefers
    thick = (any_exp & ~any_ser) | (any_exp & any_ser & ~mser);
#pragma unroll
    for (int t = 0; t < NT; t++) {
        const float ks = ke[t].x * s;
        float2 q;
        if ((thick >> t) & 1u) {
            q.x = -ks * LOC_LOG2E;
            q.y = __fdividef(ke[t].y, ke[t].x);  // source function in occupation-number units
        } else {
            q.x = ks;
            q.y = ke[t].y * s;
        }
        T.tp[g][j][t] = step ? q : make_float2(0.f, 0.f);
    }
    r.wbop |= (step ? thick : 0u) << LOC_THICK_SHIFT;
    T.rs[g][j] = r;
}

// One pass over a span of 32 channels for the four ray steps of a round: lane l8 of a group updates the quad at `sq`
// (its channels have the offsets jf[0..3] from the span start of RecS) for all NT transitions.
//   MASK = false: the common path -- no masks, the quad is known to lie inside the spectrum
//   MASK = true : channel k takes part iff m[k]; the quad is loaded / stored iff `inq`
// Accumulates the lane's partial sums a[t] += sum_k n_k X_k, b[t] += sum_k X_k, sphi += sum_k phi_k.
#define LOC_SERIES(C0, P, B2, B3, B4, B5) fma2(C0, fma2(C0, fma2(C0, fma2(C0, B5, B4), B3), B2), P)
template <int NT, bool MASK>
__device__ __forceinline__ void span_pass(float *sq, int nchp, const float2 *tpr, const RecS &rs, const float (&jf)[4], unsigned thick,
                                          unsigned any_thick, unsigned any_thin, bool inq, const bool (&m)[4], float (&a)[NT], float (&b)[NT],
                                          float &sphi)
{
    float e[4];
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const float y = fmaf(jf[k], rs.ky, rs.A);
        e[k] = ex2f(fmaf(-y, y, rs.lamp));
        if (MASK) e[k] = m[k] ? e[k] : 0.0f;
    }
    sphi += (e[0] + e[1]) + (e[2] + e[3]);
    const f32x2 P01 = pk2(e[0], e[1]), P23 = pk2(e[2], e[3]);
    const f32x2 ONE2 = pk2(1.0f, 1.0f), MONE2 = pk2(-1.0f, -1.0f);
    f32x2 B2a = 0ull, B2b = 0ull, B3a = 0ull, B3b = 0ull, B4a = 0ull, B4b = 0ull, B5a = 0ull, B5b = 0ull;
    // powers of phi for the series, shared by the transitions of the round that use it (all rays thin, or mixed)
    if ((~any_thick | any_thin) & ((1u << NT) - 1u)) {
        const f32x2 K2 = pk2(-0.5f, -0.5f), K3 = pk2(1.0f / 6.0f, 1.0f / 6.0f), K4 = pk2(-1.0f / 24.0f, -1.0f / 24.0f);
        const f32x2 s01 = mul2(P01, P01), s23 = mul2(P23, P23);
        B2a = mul2(s01, K2);
        B2b = mul2(s23, K2);
        B3a = mul2(mul2(s01, P01), K3);
        B3b = mul2(mul2(s23, P23), K3);
        B4a = mul2(mul2(s01, s01), K4);
        B4b = mul2(mul2(s23, s23), K4);
        const f32x2 K5 = pk2(-0.2f, -0.2f);
        B5a = mul2(mul2(B4a, P01), K5);
        B5b = mul2(mul2(B4b, P23), K5);
    }
    // Three phases, so that the loads and the common tail of all transitions are straight-line code the scheduler can
    // interleave (the form of X is chosen by warp-uniform branches per transition).
    float2 q[NT];
    float4 n4[NT];
#pragma unroll
    for (int t = 0; t < NT; t++) {
        q[t] = tpr[t];
        n4[t] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (!MASK || inq) n4[t] = *reinterpret_cast<const float4 *>(sq + t * nchp);
    }
    f32x2 X01[NT], X23[NT];
    float al[NT];
#pragma unroll
    for (int t = 0; t < NT; t++) {
        const f32x2 C0 = pk2(q[t].x, q[t].x);
        if (!((any_thick >> t) & 1u)) {  // every stepping ray of the warp uses the series in this transition
            X01[t] = LOC_SERIES(C0, P01, B2a, B3a, B4a, B5a);
            X23[t] = LOC_SERIES(C0, P23, B2b, B3b, B4b, B5b);
            al[t] = -q[t].x;
        } else {
            float z0, z1, z2, z3;
            upk2(mul2(C0, P01), z0, z1);
            upk2(mul2(C0, P23), z2, z3);
            const f32x2 E01 = pk2(ex2f(z0), ex2f(z1)), E23 = pk2(ex2f(z2), ex2f(z3));
            X01[t] = fma2(E01, MONE2, ONE2);
            X23[t] = fma2(E23, MONE2, ONE2);
            al[t] = -1.0f;
            if ((any_thin >> t) & 1u) {  // mixed: both forms, selected per ray
                const bool tk = (thick >> t) & 1u;
                float x0, x1, x2, x3, s0, s1, s2, s3;
                upk2(X01[t], x0, x1);
                upk2(X23[t], x2, x3);
                upk2(LOC_SERIES(C0, P01, B2a, B3a, B4a, B5a), s0, s1);
                upk2(LOC_SERIES(C0, P23, B2b, B3b, B4b, B5b), s2, s3);
                X01[t] = pk2(tk ? x0 : s0, tk ? x1 : s1);
                X23[t] = pk2(tk ? x2 : s2, tk ? x3 : s3);
                al[t] = tk ? -1.0f : -q[t].x;
            }
        }
    }
#pragma unroll
    for (int t = 0; t < NT; t++) {
        const f32x2 N01 = pk2(n4[t].x, n4[t].y), N23 = pk2(n4[t].z, n4[t].w);
        const f32x2 C1 = pk2(q[t].y, q[t].y), AL = pk2(al[t], al[t]);
        float a0, a1, b0, b1;
        upk2(fma2(N01, X01[t], mul2(N23, X23[t])), a0, a1);
        upk2(add2(X01[t], X23[t]), b0, b1);
        if (MASK) {  // several passes may follow one another
            a[t] += a0 + a1;
            b[t] += b0 + b1;
        } else {
            a[t] = a0 + a1;
            b[t] = b0 + b1;
        }
        float r0, r1, r2, r3;
        upk2(fma2(X01[t], fma2(AL, N01, C1), N01), r0, r1);
        upk2(fma2(X23[t], fma2(AL, N23, C1), N23), r2, r3);
        if (!MASK || inq) *reinterpret_cast<float4 *>(sq + t * nchp) = make_float4(r0, r1, r2, r3);
    }
}

template <int NT, bool GEOM>
__global__ void __launch_bounds__(32) k_sim3d(Sim3D P)
{
    extern __shared__ __align__(16) float smem[];
    __shared__ WarpTables<NT> T;               // separate object: no aliasing with the spectra
    const int lane = threadIdx.x, grp = lane >> 3, l8 = lane & 7;
    const int nchp = P.nchp;
    const int spec = NT * nchp;                // floats per ray spectrum
    float *sn_all = smem;                      // [4][NT][nchp]
    float *sn = sn_all + grp * spec;
    float *slots_warp = P.pool + (long long)blockIdx.x * LOC_GROUPS * P.nslot * spec;
    const float jf[4] = {(float)(4 * l8), (float)(4 * l8 + 1), (float)(4 * l8 + 2), (float)(4 * l8 + 3)};

    long long off = 0, end = 0;  // this group's position in the stream
    bool done = false;
    float d0 = 0.f, d1 = 0.f, d2 = 0.f, sf = 0.f;
    unsigned long long mysteps = 0, myactive = 0;
    uint2 nrec = make_uint2(0u, LOC_OP_NOP << 24);  // record of the next chunk, fetched one chunk ahead
    bool have_next = false;

    for (;;) {
        // ---- refill: groups whose task is exhausted take the next root ray from the queue ----
        {
            const bool need = !done && off >= end;
            long long task = 0;
            if (need && l8 == 0) task = atomicAdd(P.queue, 1u);
            task = __shfl_sync(0xffffffffu, task, grp * 8);
            if (need) {
                have_next = false;
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
        if (__all_sync(0xffffffffu, done)) break;
        // ---- prepare: lane l8 of each group decodes record off + l8 of its ray ----
        uint2 rec = make_uint2(0u, LOC_OP_NOP << 24);
        if (have_next)
            rec = nrec;
        else if (!done && off + l8 < end)
            rec = __ldg(P.stream + off + l8);
        off += LOC_CHUNK;
        have_next = !done && off < end;
        nrec = make_uint2(0u, LOC_OP_NOP << 24);
        if (have_next && off + l8 < end) nrec = __ldg(P.stream + off + l8);
        prepare_record<NT>(P, rec, d0, d1, d2, sf, T, grp, l8);
        __syncwarp();

        // ---- 8 rounds: every group consumes one record per round ----
        for (int r = 0; r < LOC_CHUNK; r++) {
            const unsigned cls = T.cls[r];
            if (cls & LOC_CLS_CTRL) {
                // spectrum operations, executed by the whole warp for one group at a time
                for (int g = 0; g < LOC_GROUPS; g++) {
                    const unsigned gop = T.opdz[g][r] >> 24, gx = T.cell[g][r];
                    float *gs = sn_all + g * spec;
                    float *slot = slots_warp + ((long long)g * P.nslot + gx) * spec;
                    if (gop == LOC_OP_BG) {
#pragma unroll
                        for (int t = 0; t < NT; t++) {
                            const float bg = P.S.bgocc[P.slot0 + t];
                            for (int c = lane; c < nchp; c += 32) gs[t * nchp + c] = bg;
                        }
                    } else if (gop == LOC_OP_SAVE) {
                        for (int i = lane * 4; i < spec; i += 128) *reinterpret_cast<float4 *>(slot + i) = *reinterpret_cast<const float4 *>(gs + i);
                    } else if (gop == LOC_OP_LOAD) {
                        for (int i = lane * 4; i < spec; i += 128) *reinterpret_cast<float4 *>(gs + i) = *reinterpret_cast<const float4 *>(slot + i);
                    }
                }
                __syncwarp();
            }
            if (!(cls & LOC_CLS_STEP)) continue;
            const unsigned any_thick = cls & 0xfffu, any_thin = (cls >> LOC_CLS_THIN_SHIFT) & 0xfffu;
            const RecS rs = T.rs[grp][r];
            const unsigned thick = (rs.wbop >> LOC_THICK_SHIFT) & 0xfffu;
            const int wb = (int)(rs.wbop & LOC_WB_MASK);
            const float2 *tpr = T.tp[grp][r];

            float a[NT], b[NT];
#pragma unroll
            for (int t = 0; t < NT; t++) a[t] = b[t] = 0.f;
            float sphi = 0.f;
            if (!(cls & LOC_CLS_SLOW)) {
                const bool nomask[4] = {true, true, true, true};
                span_pass<NT, false>(sn + wb + 4 * l8, nchp, tpr, rs, jf, thick, any_thick, any_thin, true, nomask, a, b, sphi);
            } else {
                // masked passes of 32 channels over the nominal window (several when the line is very thick)
                const int2 win = T.win[grp][r];
                int base = win.x & ~3;
                while (__any_sync(0xffffffffu, base <= win.y)) {
                    const int cb = base + 4 * l8;  // the lane's quad in this pass (win.y < nch <= nchp: in range if cb <= win.y)
                    const float ob = (float)(base - wb);
                    const float jo[4] = {jf[0] + ob, jf[1] + ob, jf[2] + ob, jf[3] + ob};
                    const bool m[4] = {cb >= win.x && cb <= win.y, cb + 1 >= win.x && cb + 1 <= win.y, cb + 2 >= win.x && cb + 2 <= win.y,
                                       cb + 3 >= win.x && cb + 3 <= win.y};
                    span_pass<NT, true>(sn + cb, nchp, tpr, rs, jo, thick, any_thick, any_thin, cb <= win.y, m, a, b, sphi);
                    base += LOC_SPAN;
                }
            }
            // ---- reduction over the 8 lanes of each group, through shared memory (no selects, DESIGN 6.4) ----
            sphi += __shfl_xor_sync(0xffffffffu, sphi, 4);
            sphi += __shfl_xor_sync(0xffffffffu, sphi, 2);
            sphi += __shfl_xor_sync(0xffffffffu, sphi, 1);
            float2 *pg = T.part[grp];
#pragma unroll
            for (int t = 0; t < NT; t++) pg[t * WarpTables<NT>::ROW + l8] = make_float2(a[t], b[t]);
            __syncwarp();
            // lane t of a group adds up row t and issues the two float atomics of (cell, transition t) as one 64-bit RED
            const bool step = rs.wbop & LOC_RS_STEP;
            const unsigned cell = T.cell[grp][r];
            const float w = T.w[grp][r];
            const float wesc = w - w * sphi;  // photons emitted outside the updated channels escape (DESIGN 5.3)
#pragma unroll
            for (int t0 = 0; t0 < NT; t0 += 8) {
                const int t = t0 + l8;
                if (step && t < NT) {
                    const float4 *row = reinterpret_cast<const float4 *>(pg + t * WarpTables<NT>::ROW);
                    const float4 r0 = row[0], r1 = row[1], r2 = row[2], r3 = row[3];
                    const f32x2 s01 = add2(add2(pk2(r0.x, r0.y), pk2(r0.z, r0.w)), add2(pk2(r1.x, r1.y), pk2(r1.z, r1.w)));
                    const f32x2 s23 = add2(add2(pk2(r2.x, r2.y), pk2(r2.z, r2.w)), add2(pk2(r3.x, r3.y), pk2(r3.z, r3.w)));
                    float A, B;
                    upk2(add2(s01, s23), A, B);
                    // scale of the sums: w for the series form, w / (kappa s) for the exponential form (c0 = -kappa s log2 e)
                    const float sc = ((thick >> t) & 1u) ? __fdividef(-LOC_LOG2E * w, tpr[t].x) : w;
                    float2 *cn = P.cnt + (long long)cell * P.nsp + P.slot0 + t;
                    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(cn), "f"(A * sc), "f"(fmaf(B, sc, wesc)) : "memory");
                }
            }
            if (step && l8 == 0) {
                mysteps++;
                if (GEOM) {
                    atomicAdd(&P.visits[cell], 1u);
                    atomicAdd(&P.pathz[cell], T.opdz[grp][r] & 0x1fffffu);
                    const float h5 = 5.0f * 0.8493218f / rs.ky, cc = (float)wb - rs.A / rs.ky;  // 5 sigma in channels, line centre
                    myactive += max(0, min(P.nch - 1, (int)floorf(cc + h5)) - max(0, (int)ceilf(cc - h5)) + 1);
                }
            }
            __syncwarp();  // the next round's quads were written by other lanes
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
    const size_t smem = sizeof(float) * LOC_GROUPS * NT * P.nchp;  // + static: the prepare tables
    if (smem > 200 * 1024 || P.nch > (int)LOC_WB_MASK) {
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
