// loc_sim3d.cu -- 3D radiative kernel: replays the precomputed step streams (loc_paths3d.cu) every ALI iteration and
// evaluates, per ray step and velocity channel, the Doppler-shifted profile, the optical depth, the photon
// transfer of Eq. 3 and the two per-cell sums (Eq. 2 first term; escape fraction of PAPER.md:81) for all traced
// transitions at once (the "all transitions in one pass" option the paper leaves open).
//
// Work decomposition (DESIGN 6.4).  A CTA of TWO warps carries FOUR rays at a time; both warps walk the same four rays in
// lock step and split the traced TRANSITIONS between them (warp 0 the first half, warp 1 the rest): the rays' spectra and
// per-step records in shared memory are shared, so twice as many warps are resident for the same shared memory, and
// each warp prepares and reduces only its own transitions.  Within a warp each ray has a quarter-warp ("group" of 8
// lanes).  Every
// step touches a SPAN of 32 consecutive channels that starts at a multiple of 4 and is centred on the Doppler-shifted
// line; lane l8 of the group owns the aligned quad  span + 4 l8 .. + 3, so that
//   * the photon spectrum of a ray lives in shared memory and is read / written with one 128-bit access per lane and
//     transition, conflict free for any span position (a quarter-warp is one shared-memory phase);
//   * the per-channel arithmetic is done on packed pairs (fma.rn.f32x2) and is ONE straight-line expression for both
//     regimes of the optical depth (below): no masks, no selects, no branches per transition;
//   * the sums over a lane's 4 channels are free, and the cross-lane reduction is a halving butterfly in registers
//     (warp_multi_reduce): lane t of the group ends up with the total of transition t and issues ONE 64-bit RED for
//     the cell's (SJ, ESC) pair;
//   * all per-step scalar work (record decode, Doppler shift, window, per-transition coefficients, scale of the sums,
//     counter offset) is done in a "prepare" phase, two lanes of each warp per record for 4 records x 4 rays at once,
//     from cell data prefetched into registers one chunk ahead, and left in one shared-memory record per (ray, round):
//     the round addresses everything with immediate offsets from one register.  Two CTA barriers per chunk of 4 rounds
//     (records complete / records free) are the only synchronisation between the two warps.
// All traced transitions (up to the shared-memory limit) go through ONE launch: the per-step overhead is paid once
// (profiles/r1_v5_sim3d_C3.md: splitting 9 transitions over 2 launches cost ~10 ms per launch on C3).
//
// Unified per-channel factor (DESIGN 5.3).  With phi the profile value of the channel,
//     X = (1 - 2^(Ce phi)) + U phi + C0 (B2 + C0 B3),   B2 = -phi^2 / 2,  B3 = phi^3 / 6
//     n' = n + X (c1 + alpha n),     a += n X,   b += X
// a ray step whose line-centre optical depth tau0 = kappa s phi_max is >= LOC_EXP_TAU uses the exponential form
// (Ce = -kappa s log2 e, U = C0 = 0, c1 = S = eps / kappa, alpha = -1: X = 1 - e^-tau), a thinner one the series
// (Ce = 0, U = 1, C0 = kappa s, c1 = eps s, alpha = -C0: X = phi f(tau), f = 1 - tau/2 + tau^2/6, truncation
// tau^3/24 < 1.2e-6; ex2(0) = 1 exactly, so the first bracket vanishes).  1 - e^-tau by ex2.approx and a subtraction
// has an absolute error of ~1e-7 per channel, i.e. < 1e-5 of the channel sums for tau0 >= 0.03.
// Reach of the span (DESIGN 5.3).  The profile is carried out to X sigma, X^2 = LOC_XCLIP^2 + 2 ln max(1, tau0m) with tau0m
// the largest line-centre optical depth of the step over ALL transitions.  The profile mass beyond the span is known
// analytically (wing_mass): it enters the escape fraction as it stands, and the photons of the span's edge channels
// stand for those of the thin wings beyond them in the absorbed-photon sum ("wing correction").  A step whose centred
// span does not reach X sigma takes two adjacent spans (WIDE round: two passes of the same code); bands narrower than
// the spans take a masked multi-pass path written as a rolled loop.  The four groups stay in lock step: every round each
// group consumes exactly one stream record (tasks are padded to whole chunks by the path builder); the rare spectrum
// operations (background, save, load) are executed by the whole warp for the group that needs them.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>

#include "loc_internal.cuh"

#define LOC_GROUPS 4  // rays per warp
#define LOC_CHUNK 4   // records per group and prepare phase (LOC_TASK_ALIGN is a multiple)
#define LOC_SPAN 32   // channels per pass: 8 lanes x one aligned float4
#define LOC_RAY_SKEW 8  // floats between the end of a ray's spectrum and the start of the next ray's, in shared memory
#define LOC_EXT 4     // wing extension: channels below and above the span that are carried to first order in tau (one per lane)

struct Sim3D {
    int nch, nchp, nsp, nslot;
    int slot0;  // first counter / coefficient slot handled by this launch (transitions may be split over launches)
    int geom;   // also accumulate the geometry counters (visits, path sums, active channels)
    float dv, xmin, xclip, xfull, inv_ndir;
    int nsel_all;  // traced transitions of the whole selection (this launch may hold a part)
    int geomact;   // count the active channel-transitions of the masked rounds (hyperfine structure: every part of a split launch)
    unsigned long long *nactive;
    HfsTab H;      // hyperfine structure of the selection's slots
    const Dir3 *dirs;
    const uint16_t *task_dir;
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

// ---- shared-memory record of one (ray, round), written by the prepare phase --------------------------------------
//   +0   float q0, q1, q2     log2 phi(channel wb + 16 + j) = q0 + j (q1 + j q2)      (j = -16 .. 15 inside the span)
//   +12  uint  wbop           bits 0..9 first channel of the span,
//                             bit 30 = spectrum operation (BG / SAVE / LOAD), bit 31 = the record is a STEP
//   +16  uint  coff           cell * nsp + slot0 : element offset of the cell's counter record (STEP); slot (SAVE / LOAD)
//   +20  float w              a s / V_eff = dzeta / (h NDIR)
//   +24  uint  opdz           opcode | level | dzeta (stream word)
//   +28  float cc             line centre in channel units
//   +32  float tm[4]          largest line-centre optical depth among the transitions of preparing lane 2 W + half
//   +48  float -, -, qe       profile mass outside the span (or -1: the round sums phi itself), 1 pad word
//   +64  float2 cf[NT]        (kappa s, c1) per transition: c1 = eps / kappa (exponential form) or eps s (series); the lowest
//                             mantissa bit of c1 holds the form (1 = exponential): make_tcoef
//   then float sc[NT4]        scale of the channel sums: w (series) or w / (kappa s) (exponential); NT4 = NT rounded up to 4
#define LOC_WB_MASK 0x3ffu
#define LOC_RS_WIDE 0x10000000u  // mode bits of a step, formed after the prepare phase (step_mode): two spans
#define LOC_RS_SLOW 0x20000000u  //   masked multi-pass path
#define LOC_RS_CTRL 0x40000000u
#define LOC_RS_STEP 0x80000000u

#define LOC_EXP_TAU 0.05f  // line-centre optical depth of a step from which the exponential form is used

template <int NT>
struct Lay {
    static constexpr int NT4 = (NT + 3) & ~3;
    static constexpr int NT0 = (NT + 1) / 2;         // transitions of warp 0; warp 1 has the other NT - NT0
    static constexpr int TM = 32;                    // byte offset of tm[]
    static constexpr int QW = 48;                    // byte offset of (ql, qh)
    static constexpr int CF = 64;                    // byte offset of cf[]: (kappa s, c1 | form bit) per transition
    static constexpr int SC = CF + 8 * NT;           // byte offset of sc[]
    static constexpr int RAW = (SC + 4 * NT4 + 15) & ~15;
    // record stride = 32 (mod 128) bytes and group stride = 16 (mod 128): the 64-bit stores of the prepare phase (4 records
    // x 2 lanes x 2 groups per half-warp) and the broadcast loads of the rounds are then free of bank conflicts
    static constexpr int RECB = RAW + (32 + 128 - RAW % 128) % 128;
    static constexpr int GSB = LOC_CHUNK * RECB + (16 + 128 - (LOC_CHUNK * RECB) % 128) % 128;
    // per-lane partial sums (a_t, b_t) of the round: [group][t][lane], rows of 10 float2 (8 used) = 80 bytes: the
    // reducing lanes of a group read 8 different rows with LDS.128 conflict free; then per warp one row of 8 floats:
    // the lanes' sums of phi.  Groups 16 banks apart.
    static constexpr int ROWB = 80;
    static constexpr int PHI = NT * ROWB;            // + 32 * warp
    static constexpr int PW0 = (NT * ROWB + 64) / 4;
    static constexpr int PGB = 4 * (PW0 + ((16 + 32 - PW0 % 32) % 32));
    static constexpr int OFF_REC = 0;                                  // relative to the table base
    static constexpr int OFF_CLS = OFF_REC + LOC_GROUPS * GSB;         // class word of each round of the chunk
    static constexpr int OFF_TASK = OFF_CLS + 4 * LOC_CHUNK;           // task taken from the queue, per group
    static constexpr int OFF_PART = OFF_TASK + 4 * LOC_GROUPS;
    static constexpr int BYTES = OFF_PART + LOC_GROUPS * PGB;
};

// ---- shared memory through 32-bit addresses with immediate offsets ------------------------------------------------
__device__ __forceinline__ float rcpf(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float4 ldg_keep(const float *p, unsigned long long pol)
{
    float4 v;
    asm volatile("ld.global.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ void stg_keep(float *p, float4 v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
template <int OFF = 0>
__device__ __forceinline__ float4 lds128(unsigned a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF = 0>
__device__ __forceinline__ uint4 lds128u(unsigned a)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4+%5];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF = 0>
__device__ __forceinline__ float lds32(unsigned a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF = 0>
__device__ __forceinline__ unsigned lds32u(unsigned a)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF = 0>
__device__ __forceinline__ float2 lds64(unsigned a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+%3];" : "=f"(v.x), "=f"(v.y) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF = 0>
__device__ __forceinline__ void sts128(unsigned a, float4 v)
{
    asm volatile("st.shared.v4.f32 [%0+%1], {%2, %3, %4, %5};" ::"r"(a), "n"(OFF), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
template <int OFF = 0>
__device__ __forceinline__ void sts128u(unsigned a, uint4 v)
{
    asm volatile("st.shared.v4.u32 [%0+%1], {%2, %3, %4, %5};" ::"r"(a), "n"(OFF), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
template <int OFF = 0>
__device__ __forceinline__ void sts64(unsigned a, float2 v)
{
    asm volatile("st.shared.v2.f32 [%0+%1], {%2, %3};" ::"r"(a), "n"(OFF), "f"(v.x), "f"(v.y) : "memory");
}
template <int OFF = 0>
__device__ __forceinline__ void sts32(unsigned a, float v)
{
    asm volatile("st.shared.f32 [%0+%1], %2;" ::"r"(a), "n"(OFF), "f"(v) : "memory");
}
template <int OFF = 0>
__device__ __forceinline__ void sts32u(unsigned a, unsigned v)
{
    asm volatile("st.shared.u32 [%0+%1], %2;" ::"r"(a), "n"(OFF), "r"(v) : "memory");
}



// Profile mass below channel s0 and above channel s0 + len - 1 for a line centred at channel cc with 1 / sigma = rs (per
// channel): Q(x) = phi(x) / (x + 1/(x + 2/(x + 3/(x + 4/x)))), good to ~1e-5 of Q for the distances x >= 3 sigma that
// occur; `far` = both distances are.  Their sum is 1 - sum phi over the channels s0 .. s0 + len - 1, far more accurate
// than that difference in float32 (the escape fraction of a thick cell is ~1e-3).
__device__ __forceinline__ void wing_mass(float cc, float rs, float s0, float len, float &Ql, float &Qh, bool &far)
{
    const float xl = (cc - (s0 - 0.5f)) * rs, xh = ((s0 + len - 0.5f) - cc) * rs;
    // the continued fraction written as one rational function: x + 1/(x + 2/(x + 3/(x + 4/x))) = x (u^2 + 10 u + 15) / (u^2 + 9 u + 8),
    // u = x^2: one reciprocal per side instead of a chain of five
    const float ul = xl * xl, uh = xh * xh;
    Ql = 0.3989422804f * ex2f(-0.7213475f * ul) * fmaf(ul, ul + 9.0f, 8.0f) * rcpf(xl * fmaf(ul, ul + 10.0f, 15.0f));
    Qh = 0.3989422804f * ex2f(-0.7213475f * uh) * fmaf(uh, uh + 9.0f, 8.0f) * rcpf(xh * fmaf(uh, uh + 10.0f, 15.0f));
    far = xl >= 3.0f && xh >= 3.0f;
}

// Split of the transitions: warp W of the CTA owns transitions TB .. TB + NW - 1; lane `half` (0 / 1) of a record's lane
// pair prepares NHW of them, from T0(half).
template <int NT, int W>
struct Own {
    // W = 2: the CTA is ONE warp that owns every transition (small NT: no second warp repeating the stream fetch, the
    // prepare phase and the barriers for one or two transitions; profiles/r2_sim3d.md)
    static constexpr bool ONE = W == 2;
    static constexpr int TB = ONE ? 0 : (W ? Lay<NT>::NT0 : 0);
    static constexpr int NW = ONE ? NT : (W ? NT - Lay<NT>::NT0 : Lay<NT>::NT0);
    static constexpr int NHW = (NW + 1) / 2;
    static constexpr int NHR = NHW > 0 ? NHW : 1;  // array sizes
    // the warp with fewer transitions also prepares the record headers, keeps the statistics and the geometry counters
    static constexpr int HW = (NT - Lay<NT>::NT0 > 0 && NT - Lay<NT>::NT0 < Lay<NT>::NT0) ? 1 : 0;
    static constexpr bool HEAD = ONE || W == HW;
    static constexpr int TMI = ONE ? 0 : 2 * W;  // first of the warp's two slots of tm[]
};

// Cell data of one stream record as the prepare phase needs it: the kinematics and the (kappa, eps) pairs of the lane's
// transitions.
template <int NT, int W>
struct CellRegs {
    float4 kin;
    float2 cf[Own<NT, W>::NHR];
};

template <int NT, int W>
__device__ __forceinline__ void load_cell(const Sim3D &P, uint2 rec, int half, CellRegs<NT, W> &C)
{
    typedef Own<NT, W> O;
    if ((rec.y >> 24) != LOC_OP_STEP) return;
    C.kin = __ldg(P.kin + rec.x);
    const float2 *cf = P.coef + (long long)rec.x * P.nsp + P.slot0 + O::TB + half * O::NHW;
#pragma unroll
    for (int i = 0; i < O::NHW; i++)
        if (half * O::NHW + i < O::NW) C.cf[i] = __ldg(cf + i);
}

// Prepare phase: lanes (g, 2 j) and (g, 2 j + 1) of each warp decode record j of the chunk of group g; every lane fills
// the coefficients of its own transitions in the record at `rb`, lane half 0 of the header warp (Own::HEAD) also the header.  Returns the
// record's flag bits (LOC_RS_*).  `nact` = number of channels within 5 sigma of the line centre (the counting rule of
// the metric) for STEP records when the geometry counters are on.
template <int NT, int W>
__device__ __forceinline__ unsigned prepare_record(const Sim3D &P, uint2 rec, const CellRegs<NT, W> &C, float4 dir, unsigned rb, int half,
                                                   int &nact)
{
    typedef Lay<NT> L;
    typedef Own<NT, W> O;
    const unsigned op = rec.y >> 24;
    const bool step = op == LOC_OP_STEP;
    unsigned flags = (op == LOC_OP_BG || op == LOC_OP_SAVE || op == LOC_OP_LOAD) ? LOC_RS_CTRL : 0u;
    float s = 0.f, w = 0.f, amp = 0.f;
    float4 k = make_float4(0.f, 0.f, 0.f, 1.f);
    if (step) {
        k = C.kin;
        const unsigned dz = rec.y & 0x1fffffu;
        const int lev = (rec.y >> 21) & 7;
        s = (float)dz * dir.w;
        w = (float)dz * P.inv_ndir * __int_as_float((127 - LOC_LB + lev) << 23);
        amp = P.dv * 0.3989422804f * rcpf(k.w);
        flags |= LOC_RS_STEP;
    }
    nact = 0;
    if (O::HEAD && half == 0) {
        float q0 = -INFINITY, q1 = 0.f, q2 = 0.f, cc = 0.f, ql = 0.f, qh = 0.f, qe = -1.f;  // phi = 2^(-inf) = 0 for records that are not steps
        unsigned wb = 0u;
        if (step) {
            const float v0 = -(k.x * dir.x + k.y * dir.y + k.z * dir.z);  // DESIGN R6
            const float inv_dv = rcpf(P.dv);
            cc = fmaf(v0, inv_dv, 0.5f * (float)(P.nch - 1));  // line centre in channel units
            const float sigch = k.w * inv_dv;
            // the span: 32 channels from a multiple of 4, centred on the line, inside the band (whether it serves the
            // step is decided by step_mode, once the optical depths of all transitions are known)
            const int wbmax = (P.nch - LOC_SPAN) & ~3;
            int iwb = 4 * (int)rintf((cc - 15.5f) * 0.25f);
            iwb = max(0, min(iwb, wbmax));
            if (P.nch < LOC_SPAN) iwb = 0;
            // log2 phi(channel wb + 16 + j) = lamp - (A + j ky)^2 with A = (wb + 16 - cc) ky: the quadratic in j is
            // expanded around the middle of the span, where |A| is a few channels only
            const float ky = 0.8493218f * rcpf(sigch);  // sqrt(log2(e) / 2) in channel units
            const float A = ((float)(iwb + 16) - cc) * ky;
            q0 = fmaf(-A, A, __log2f(amp));
            q1 = -2.0f * A * ky;
            q2 = -ky * ky;
            wb = (unsigned)iwb;
            // qe = profile mass outside the span (-1: the round takes 1 - sum phi)
            {
                float Ql, Qh;
                bool far;
                wing_mass(cc, rcpf(sigch), (float)iwb, (float)LOC_SPAN, Ql, Qh, far);
                // channels wider than the line: the sum of the sampled profile differs from its integral (by e^{-2 pi^2
                // (sigma/dv)^2}: 3e-9 at sigma = dv, 7e-3 at sigma = dv/2), so the analytic wing mass does not stand for
                // 1 - sum phi any more: the round then takes the sum itself (DESIGN 5.3)
                far = far && sigch >= 1.0f;
                qe = far ? Ql + Qh : -1.0f;
            }
            if (__builtin_expect(P.geom != 0, 0)) nact = max(0, min(P.nch - 1, (int)floorf(cc + 5.0f * sigch)) - max(0, (int)ceilf(cc - 5.0f * sigch)) + 1);
        }
        sts128u(rb, make_uint4(__float_as_uint(q0), __float_as_uint(q1), __float_as_uint(q2), wb | flags));
        const unsigned coff = step ? rec.x * (unsigned)P.nsp + (unsigned)P.slot0 : rec.x;
        sts128u(rb + 16, make_uint4(coff, __float_as_uint(w), rec.y, __float_as_uint(cc)));
        sts128(rb + L::QW, make_float4(ql, qh, qe, 0.f));
        if (O::ONE) sts64(rb + L::TM + 8, make_float2(0.f, 0.f));  // the slots of the absent second warp
    }
    // per transition, branch free: the exponential form from tau0 >= LOC_EXP_TAU (header comment); records that are not
    // steps have kappa = eps = s = w = 0 and get all-zero coefficients
    const float wos = w * rcpf(s);  // not used when s = 0
    float tm = 0.f;
#pragma unroll
    for (int i = 0; i < O::NHW; i++) {
        if (half * O::NHW + i < O::NW) {
            const int t = O::TB + half * O::NHW + i;
            const float2 ke = step ? C.cf[i] : make_float2(0.f, 0.f);
            const float ks = ke.x * s;
            const float tau0 = fabsf(ks) * amp;
            tm = fmaxf(tm, tau0);
            const bool thick = tau0 >= LOC_EXP_TAU;
            const float rk = rcpf(ke.x);
            const float c1 = thick ? ke.y * rk : ke.y * s;  // source function in occupation-number units | eps s
            sts64(rb + L::CF + 8 * t, make_float2(ks, __uint_as_float((__float_as_uint(c1) & ~1u) | (thick ? 1u : 0u))));
            sts32(rb + L::SC + 4 * t, thick ? wos * rk : w);  // the sums of the exponential form carry a factor kappa s
        }
    }
    sts32(rb + L::TM + 4 * (O::TMI + half), tm);
    return flags;
}

// first channel of the pair of spans (64 channels from a multiple of 4, centred on the line, inside the band) of a WIDE step
__device__ __forceinline__ int wide_start(int nch, float cc)
{
    const int wmax = (nch - 2 * LOC_SPAN) & ~3;
    return max(0, min(4 * (int)rintf((cc - 31.5f) * 0.25f), wmax));
}

// Mode of a ray step, formed by one lane per record after the prepare phase of both warps (the largest line-centre
// optical depth tau0m of ALL transitions is needed): the profile must be carried out to X sigma with
// X^2 = LOC_XCLIP^2 + 2 ln max(1, tau0m), so that the mass left outside stays the same fraction of the step's escape
// sum  sum phi f(tau) ~ 1 / tau0  as LOC_XCLIP sigma for a thin line (DESIGN 5.3).  If the centred 32-channel span reaches
// that far on both sides (or to the edge of the band) the step is a common round; else, if two adjacent spans do, a WIDE
// round (two passes); else a masked round over its exact window.  Returns the record's flags with the mode bits.
// WIDEP: the kernel has the two-span (WIDE) round; without it such steps take the masked round (see k_sim3d)
template <int NT, bool HFS, bool WIDEP>
__device__ __forceinline__ unsigned step_mode(const Sim3D &P, unsigned rb, float &qe_wide)
{
    qe_wide = -1.0f;  // profile mass outside the pair of spans of a WIDE step (-1: the round takes 1 - sum phi)
    typedef Lay<NT> L;
    const float4 h0 = lds128(rb);
    const unsigned wbop = __float_as_uint(h0.w);
    unsigned flags = wbop & (LOC_RS_STEP | LOC_RS_CTRL);
    if (wbop & LOC_RS_STEP) {
        const float4 tm = lds128(rb + L::TM);
        const float cc = lds32(rb + 28);
        const float tau0m = fmaxf(fmaxf(tm.x, tm.y), fmaxf(tm.z, tm.w));
        const float lt = tau0m > 1.0f ? 1.3862944f * __log2f(tau0m) : 0.0f;  // 2 ln max(1, tau0m)
        const float X2 = fmaf(P.xclip, P.xclip, lt);
        float need;  // X sigma in channels = sqrt(X2) * 0.8493218 / sqrt(-q2)
        asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(need) : "f"(X2 * 0.7213475f * rcpf(-h0.z)));
        // ... and the span with its wing extension must reach X_f sigma, X_f^2 = xfull^2 + 2 ln max(1, tau0m)
        float needf;
        asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(needf) : "f"(fmaf(P.xfull, P.xfull, lt) * 0.7213475f * rcpf(-h0.z)));
        const int wb = (int)(wbop & LOC_WB_MASK);
        const bool ok1 = P.nch >= LOC_SPAN && (wb == 0 || cc - (float)wb >= need) && (wb + LOC_SPAN >= P.nch || (float)(wb + LOC_SPAN - 1) - cc >= need) &&
                         (wb - LOC_EXT <= 0 || cc - (float)(wb - LOC_EXT) >= needf) &&
                         (wb + LOC_SPAN + LOC_EXT >= P.nch || (float)(wb + LOC_SPAN + LOC_EXT - 1) - cc >= needf);
        if (-h0.z > 0.7213475f || HFS) {
            // channels wider than the line (sigma < dv; -q2 = log2(e) / (2 sigch^2)): the exact masked path, which sums the
            // sampled profile itself and evaluates it from the distance to the line centre (DESIGN 5.3); so do all steps of a
            // model with hyperfine structure (a profile per transition, components spread over the band)
            flags |= LOC_RS_SLOW;
        } else if (__builtin_expect(!ok1, 0)) {
            const int ww = wide_start(P.nch, cc);
            const float need2 = fmaxf(need, needf);  // a pair of spans has no extension
            const bool ok2 = P.nch >= 2 * LOC_SPAN && (ww == 0 || cc - (float)ww >= need2) && (ww + 2 * LOC_SPAN >= P.nch || (float)(ww + 2 * LOC_SPAN - 1) - cc >= need2);
            flags |= (WIDEP && ok2) ? LOC_RS_WIDE : LOC_RS_SLOW;
            if (ok2) {
                float Ql, Qh;
                bool far;
                wing_mass(cc, 1.1774100f * sqrtf(-h0.z), (float)ww, (float)(2 * LOC_SPAN), Ql, Qh, far);
                if (far && -h0.z <= 0.7213475f) qe_wide = Ql + Qh;  // -q2 = log2(e) / (2 sigch^2): sigch >= 1 as in prepare_record
            }
        }
    }
    return flags;
}

// Coefficients of one (ray step, transition) for the unified per-channel factor (header comment), derived by every lane
// from the record's pair cf = (kappa s, c1) -- c1 = eps / kappa (exponential form) or eps s (series), the form in the
// lowest mantissa bit of c1 (one ulp) -- instead of being read as six floats: the kernel is bound by shared-memory
// wavefronts (profiles/r2_sim3d.md), a 64-bit broadcast load is 2 of them where LDS.128 + LDS.32 were 5.
struct TCoef {
    float C0, Ce, c1, al, U, g, ks, es;  // g = unit of the channel sums relative to phi n: kappa s (exponential) or 1 (series)
};
__device__ __forceinline__ TCoef make_tcoef(float2 cf)
{
    TCoef c;
    const bool thick = __float_as_uint(cf.y) & 1u;
    c.ks = cf.x;
    c.c1 = cf.y;
    c.C0 = thick ? 0.0f : cf.x;
    c.Ce = thick ? -LOC_LOG2E * cf.x : 0.0f;
    c.al = thick ? -1.0f : -cf.x;
    c.U = thick ? 0.0f : 1.0f;
    c.g = thick ? cf.x : 1.0f;
    c.es = cf.y * c.g;  // eps s: the first-order emission of the wing-extension channel
    return c;
}

// Masked multi-pass round for one lane's ray step (rare: DESIGN 6.4): passes of 32 channels over the step's nominal
// window [clo, chi], which is formed here from the record (the largest line-centre optical depth of ALL transitions sets
// its width, DESIGN 5.3), for the warp's own transitions.  Leaves the lane's partial sums in its slots of the `part` rows:
// (a_t, b_t - g_t sum phi), i.e. with the lane's sum of the sampled profile already folded into b (see the reduction).
// Scalar arithmetic, rolled over the transitions; same expressions as the common round.
// HFS: the model has hyperfine structure (a template parameter: the kernels of models without it carry none of that code --
// the instruction-fetch stalls of the common round grow with the size of the loop body, profiles/r2_sim3d.md)
template <int NT, int W, bool HFS>
__device__ __forceinline__ unsigned slow_round(const Sim3D &P, unsigned rb, unsigned sqg, unsigned pl, int l8, int nchp)
{
    typedef Lay<NT> L;
    typedef Own<NT, W> O;
    const float4 h0 = lds128(rb);
    const uint4 h1 = lds128u(rb + 16);
    const unsigned wbop = __float_as_uint(h0.w);
    constexpr bool hfs = HFS;  // hyperfine structure: a profile per transition, summed over its components (loc_set_hyperfine)
    int clo = 1, chi = 0;
    // the profile from the distance to the line centre: log2 phi(c) = lamp - ((c - cc) ky)^2.  (The quadratic around the
    // middle of the span that the common round uses cancels badly when the span is clamped far from the line AND the
    // channels are wide: ky ~ 8 per channel at dv = 10 sigma.)
    const float kyc = sqrtf(-h0.z), ccc = __uint_as_float(h1.w);
    const float lamp = (wbop & LOC_RS_STEP) ? __log2f(0.4697186f * kyc) : -INFINITY;
    if (wbop & LOC_RS_STEP) {
        const float ky = sqrtf(-h0.z);
        const float sigch = 0.8493218f * rcpf(ky);
        const float4 tm = lds128(rb + L::TM);
        const float tau0m = fmaxf(fmaxf(tm.x, tm.y), fmaxf(tm.z, tm.w));
        float X2 = fmaxf(P.xmin, P.xfull) * fmaxf(P.xmin, P.xfull);
        // channels wider than the line: a handful of channels whatever the reach, and no analytic wing mass on this path:
        // reach 6.5 sigma at least, + 2 ln (dv/sigma)^2 (see loc_sim1d.cu)
        if (sigch < 1.0f) X2 = fmaf(-4.0f, __logf(sigch), fmaxf(X2, 42.25f));
        if (tau0m > 1.0f) X2 = fmaf(2.0f, __logf(tau0m), X2);
        const float X = sqrtf(X2);
        const float cc = __uint_as_float(h1.w), hw = X * sigch;
        clo = max(0, (int)ceilf(cc + P.H.lo - hw));  // (lo = hi = 0 without hyperfine structure: one window for all components)
        chi = min(P.nch - 1, (int)floorf(cc + P.H.hi + hw));
    }
#pragma unroll 1
    for (int t = O::TB; t < O::TB + O::NW; t++) sts64(pl + t * L::ROWB, make_float2(0.f, 0.f));
    float sphi = 0.f;
    unsigned nact = 0;
    int base = clo & ~3;
    while (__any_sync(0xffffffffu, base <= chi)) {
        const int cb = base + 4 * l8;
        float e[4];
        bool inq = false;
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const int c = cb + k;
            const bool m = c >= clo && c <= chi;
            const float y = ((float)c - ccc) * kyc;
            e[k] = m ? ex2f(fmaf(-y, y, lamp)) : 0.0f;
            inq |= m;
        }
        sphi += (e[0] + e[1]) + (e[2] + e[3]);
        if (inq) {
#pragma unroll 1
            for (int t = O::TB; t < O::TB + O::NW; t++) {
                const TCoef tc = make_tcoef(lds64(rb + L::CF + 8 * t));
                float fold = 0.0f;
                if (hfs) {  // the transition's own profile over the same channels; its sum is folded into b here
                    const int slot = P.slot0 + t;
                    bool act[4] = {false, false, false, false};
#pragma unroll
                    for (int k = 0; k < 4; k++) e[k] = 0.0f;
                    for (int q = 0; q < P.H.nc[slot]; q++) {
                        const float wq = P.H.w[slot][q], dq = P.H.dch[slot][q];
#pragma unroll
                        for (int k = 0; k < 4; k++) {
                            const int c = cb + k;
                            const float y = ((float)c - ccc - dq) * kyc;
                            if (c >= clo && c <= chi) {
                                e[k] = fmaf(wq, ex2f(fmaf(-y, y, lamp)), e[k]);
                                act[k] |= y * y <= 18.033688f;  // within 5 sigma of the component (the metric's counting rule)
                            }
                        }
                    }
                    fold = tc.g * ((e[0] + e[1]) + (e[2] + e[3]));
                    if (P.geomact) nact += (unsigned)act[0] + (unsigned)act[1] + (unsigned)act[2] + (unsigned)act[3];
                }
                const unsigned sa = sqg + 4 * base + 4 * t * nchp;
                const float4 n4 = lds128(sa);
                float n[4] = {n4.x, n4.y, n4.z, n4.w};
                float a = 0.f, b = 0.f;
#pragma unroll
                for (int k = 0; k < 4; k++) {
                    const float p = e[k];
                    const float X = fmaf(tc.C0, fmaf(tc.C0, p * p * p * (1.0f / 6.0f), -0.5f * p * p), fmaf(tc.U, p, 1.0f - ex2f(tc.Ce * p)));
                    a = fmaf(n[k], X, a);
                    b += X;
                    n[k] = fmaf(X, fmaf(tc.al, n[k], tc.c1), n[k]);
                }
                sts128(sa, make_float4(n[0], n[1], n[2], n[3]));
                const float2 pv = lds64(pl + t * L::ROWB);
                sts64(pl + t * L::ROWB, make_float2(pv.x + a, pv.y + b - fold));
            }
        }
        base += LOC_SPAN;
    }
    if (!hfs) {
#pragma unroll 1
        for (int t = O::TB; t < O::TB + O::NW; t++) {  // fold the lane's sum of phi into b (the round sums phi itself: qe = -1)
            const TCoef tc = make_tcoef(lds64(rb + L::CF + 8 * t));
            const float2 pv = lds64(pl + t * L::ROWB);
            sts64(pl + t * L::ROWB, make_float2(pv.x, fmaf(-tc.g, sphi, pv.y)));
        }
    }
    return nact;
}

// The common round: one pass over the span for the warp's NW transitions, straight-line code.  `sq` = shared address of
// the lane's quad in transition 0, `rowb` = bytes between the spectra of consecutive transitions.  The lane's partial
// sums (a_t, b_t) are ADDED to ab[] (registers): a second pass of a WIDE round accumulates.
// fold: 1 if the round sums the sampled profile itself for the escape fraction (no analytic wing mass: qe < 0), else 0:
//       b_t -= g_t fold sum_lane(phi), so that sc_t sum_lanes(b_t) = w (sum phi f - sum phi) and the escape fraction is
//       w + that (the reduction needs no separate sum of phi).
// Wing extension (header comment): `se` = shared address (transition 0) of the lane's channel beyond the span, pe its
// profile value, `ext` = the channel exists (inside the band, and the ray takes the extension in this pass); without it
// se points at readable memory, pe = 0 and nothing is stored.
template <int NT, int W>
__device__ __forceinline__ void fast_round(unsigned rb, unsigned sq, int rowb, const float4 h0, const f32x2 J01, const f32x2 J23, unsigned se, float pe,
                                           bool ext, float fold, float2 (&ab)[Own<NT, W>::NHR * 2])
{
    typedef Lay<NT> L;
    typedef Own<NT, W> O;
    // profile: log2 phi = q0 + j (q1 + j q2)
    const f32x2 Q0 = pk2(h0.x, h0.x), Q1 = pk2(h0.y, h0.y), Q2 = pk2(h0.z, h0.z);
    float y0, y1, y2, y3;
    upk2(fma2(J01, fma2(J01, Q2, Q1), Q0), y0, y1);
    upk2(fma2(J23, fma2(J23, Q2, Q1), Q0), y2, y3);
    const f32x2 P01 = pk2(ex2f(y0), ex2f(y1)), P23 = pk2(ex2f(y2), ex2f(y3));
    float sa, sb;
    upk2(add2(P01, P23), sa, sb);
    const float sphif = (sa + sb) * fold;
    const f32x2 ONE2 = pk2(1.0f, 1.0f), MONE2 = pk2(-1.0f, -1.0f);
    const f32x2 K2 = pk2(-0.5f, -0.5f), K3 = pk2(1.0f / 6.0f, 1.0f / 6.0f);
    const f32x2 s01 = mul2(P01, P01), s23 = mul2(P23, P23);
    const f32x2 B2a = mul2(s01, K2), B2b = mul2(s23, K2);
    const f32x2 B3a = mul2(mul2(s01, P01), K3), B3b = mul2(mul2(s23, P23), K3);
    // three phases (all loads, arithmetic, all stores): the shared-memory accesses are ordered among themselves, the
    // arithmetic of the transitions in between is free to interleave
    float4 n4[O::NHR * 2];
    float2 cf[O::NHR * 2];
    float ne[O::NHR * 2];
#pragma unroll
    for (int i = 0; i < O::NW; i++) {
        cf[i] = lds64(rb + L::CF + 8 * (O::TB + i));
        n4[i] = lds128(sq + (O::TB + i) * rowb);
        ne[i] = lds32(se + (O::TB + i) * rowb);
    }
#pragma unroll
    for (int i = 0; i < O::NW; i++) {
        const TCoef tc = make_tcoef(cf[i]);
        const f32x2 C0 = pk2(tc.C0, tc.C0), CE = pk2(tc.Ce, tc.Ce), C1 = pk2(tc.c1, tc.c1), AL = pk2(tc.al, tc.al), UU = pk2(tc.U, tc.U);
        float z0, z1, z2, z3;
        upk2(mul2(CE, P01), z0, z1);
        upk2(mul2(CE, P23), z2, z3);
        const f32x2 E01 = pk2(ex2f(z0), ex2f(z1)), E23 = pk2(ex2f(z2), ex2f(z3));
        const f32x2 X01 = fma2(C0, fma2(C0, B3a, B2a), fma2(UU, P01, fma2(E01, MONE2, ONE2)));
        const f32x2 X23 = fma2(C0, fma2(C0, B3b, B2b), fma2(UU, P23, fma2(E23, MONE2, ONE2)));
        const f32x2 N01 = pk2(n4[i].x, n4[i].y), N23 = pk2(n4[i].z, n4[i].w);
        float a0, a1, b0, b1;
        upk2(fma2(N01, X01, mul2(N23, X23)), a0, a1);
        upk2(add2(X01, X23), b0, b1);
        // the wing channel: absorbed-photon sum in the units of the span's sum (g phi n), photons to first order in tau:
        // n' = n + phi (eps s - kappa s n)
        const float pg = pe * tc.g;
        ab[i].x += fmaf(pg, ne[i], a0 + a1);
        ab[i].y += fmaf(-tc.g, sphif, b0 + b1);
        ne[i] = fmaf(pe, fmaf(-tc.ks, ne[i], tc.es), ne[i]);
        upk2(fma2(X01, fma2(AL, N01, C1), N01), n4[i].x, n4[i].y);
        upk2(fma2(X23, fma2(AL, N23, C1), N23), n4[i].z, n4[i].w);
    }
#pragma unroll
    for (int i = 0; i < O::NW; i++) {
        sts128(sq + (O::TB + i) * rowb, n4[i]);
        if (ext) sts32(se + (O::TB + i) * rowb, ne[i]);
    }
}

template <int W>
__device__ __forceinline__ void cta_sync()  // both warps of the CTA (one-warp CTAs: the warp)
{
    if (W == 2)
        __syncwarp();
    else
        asm volatile("bar.sync 0, 64;" ::: "memory");
}

// One warp of the CTA.  NCHP_T: spectrum row length in floats when known at compile time (immediate offsets), 0 = P.nchp
template <int NT, int NCHP_T, int W, bool HFS>
__device__ __forceinline__ void run_warp(const Sim3D &P, float *smem)
{
    typedef Lay<NT> L;
    typedef Own<NT, W> O;
    const int lane = threadIdx.x & 31, grp = lane >> 3, l8 = lane & 7, rj = l8 >> 1, half = l8 & 1;
    const int nchp = NCHP_T ? NCHP_T : P.nchp;
    const int spec = NT * nchp;                // floats per ray spectrum
    const int specs = spec + LOC_RAY_SKEW;     // ... and between the rays' spectra in shared memory: the rays start 8 banks apart, so
                                               // that the 32-bit accesses of the wing extension of rays with the same span do not collide
    const int rowb = 4 * nchp;
    float *sn_all = smem;
    const unsigned sm0 = (unsigned)__cvta_generic_to_shared(smem);
    const unsigned tb = sm0 + 4u * LOC_GROUPS * specs;
    const unsigned rec_g = tb + L::OFF_REC + grp * L::GSB;
    const unsigned part_g = tb + L::OFF_PART + grp * L::PGB;
    const unsigned pl = part_g + 8 * l8;                        // my slot in row 0
    const unsigned sq_r = sm0 + 4u * grp * specs;   // the ray's spectrum, channel 0 of transition 0
    const unsigned sq_g = sq_r + 16 * l8;          // ... the lane's quad of a span that starts at channel 0
    const int e0 = l8 < 4 ? l8 - LOC_EXT : l8 + LOC_SPAN - LOC_EXT;  // the lane's wing-extension channel, relative to the span start
    const float je = (float)(e0 - 16);
    // the lane that owns the totals of the warp's own-th transition after the butterfly reduction of a round (-1: none)
    int own;
    {
        float dz[O::NHR * 2];
#pragma unroll
        for (int i = 0; i < O::NHR * 2; i++) dz[i] = 0.0f;
        int ob = 0, onv = O::NW;
        MultiReduce<O::NW, 4>::run(dz, lane, ob, onv);
        own = onv >= 1 ? ob : -1;
    }
    float *slots_warp = P.pool + (long long)blockIdx.x * LOC_GROUPS * P.nslot * spec;
    const float jb = (float)(4 * l8 - 16);
    const f32x2 J01 = pk2(jb, jb + 1.0f), J23 = pk2(jb + 2.0f, jb + 3.0f);
    float2 *const cnt_o = P.cnt + O::TB + (own >= 0 ? own : 0);
    // the spectrum slots of the resident CTAs (donor spectra, DESIGN 6.3) are re-read by every ray born from them: keep
    // them in L2 against the streaming traffic of the step records, coefficients and counters
    unsigned long long pol_keep;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
    const uint2 NOPREC = make_uint2(0u, LOC_OP_NOP << 24);
    const int row0 = O::TB * nchp, rown = O::NW * nchp;  // my rows of a spectrum, in floats

    long long off = 0, end = 0;  // this group's position in the stream (first record of the current chunk)
    bool done = false, fresh = false;
    float4 dir = make_float4(0.f, 0.f, 0.f, 0.f);  // (d0, d1, d2, sf) of the group's ray
    unsigned mysteps = 0;
    unsigned long long myactive = 0, hfsact = 0;
    // software pipeline over chunks: r0 = records of this chunk, r1 / r2 = of the next two (r2 in flight), `cell` = cell
    // data of r0's record, loaded during the previous chunk's rounds
    uint2 r0 = NOPREC, r1 = NOPREC, r2 = NOPREC;
    CellRegs<NT, W> cell;
    cell.kin = make_float4(0.f, 0.f, 0.f, 1.f);
#pragma unroll
    for (int i = 0; i < O::NHR; i++) cell.cf[i] = make_float2(0.f, 0.f);

    for (;;) {
        // ---- refill: groups whose task is exhausted take the next root ray from the queue (warp 0 asks, both read) ----
        const bool need = !done && off >= end;
        if (W != 1 && need && l8 == 0) sts32u(tb + L::OFF_TASK + 4 * grp, atomicAdd(P.queue, 1u));
        cta_sync<W>();  // the previous chunk's records are free; the tasks are posted
        if (__builtin_expect(need, 0)) {
            const long long task = lds32u(tb + L::OFF_TASK + 4 * grp);
            if (task >= P.ntask) {
                done = true;
                r0 = r1 = r2 = NOPREC;
            } else {
                const Dir3 *Dp = P.dirs + P.task_dir[task];
                dir = make_float4(__ldg(&Dp->d[0]), __ldg(&Dp->d[1]), __ldg(&Dp->d[2]), __ldg(&Dp->sf));
                off = __ldg(P.task_off + task);
                end = __ldg(P.task_off + task + 1);
                fresh = true;
            }
        }
        if (__all_sync(0xffffffffu, done)) break;  // the same in both warps
        if (__builtin_expect(fresh, 0)) {  // first chunk of a ray: nothing was prefetched
            r0 = __ldg(P.stream + off + rj);
            r1 = (off + LOC_CHUNK < end) ? __ldg(P.stream + off + LOC_CHUNK + rj) : NOPREC;
            load_cell<NT, W>(P, r0, half, cell);
            fresh = false;
        }
        r2 = (!done && off + 2 * LOC_CHUNK < end) ? __ldg(P.stream + off + 2 * LOC_CHUNK + rj) : NOPREC;
        // ---- prepare: lane pair rj of each group decodes record off + rj of its ray ----
        int nact;
        unsigned flags = prepare_record<NT, W>(P, r0, cell, dir, rec_g + rj * L::RECB, half, nact);
        if (O::HEAD && half == 0) {
            mysteps += flags >> 31;
            myactive += nact;
        }
        load_cell<NT, W>(P, r1, half, cell);  // for the next chunk (NOP records load nothing)
        cta_sync<W>();  // the records of the chunk are complete
        // mode of record rj (the lanes of a pair agree), then the class of round rj: OR over the four groups
        float myqew;
        const unsigned myflags = step_mode<NT, HFS, W == 2>(P, rec_g + rj * L::RECB, myqew);
        unsigned orflags = myflags | __shfl_xor_sync(0xffffffffu, myflags, 8);
        orflags |= __shfl_xor_sync(0xffffffffu, orflags, 16);

        // ---- LOC_CHUNK rounds: every group consumes one record per round ----
#pragma unroll 1
        for (int r = 0; r < LOC_CHUNK; r++) {
            const unsigned cls = __shfl_sync(0xffffffffu, orflags, 2 * r);
            const unsigned mode = __shfl_sync(0xffffffffu, myflags, 8 * grp + 2 * r);
            const float qew = __shfl_sync(0xffffffffu, myqew, 8 * grp + 2 * r);
            const unsigned rb = rec_g + r * L::RECB;
            if (__builtin_expect((cls & LOC_RS_CTRL) != 0, 0)) {
                // spectrum operations on the warp's own rows, executed by the whole warp for one group at a time; only the
                // groups that have one are visited (their lanes hold the record's CTRL bit in `mode`)
                unsigned cm = __ballot_sync(0xffffffffu, mode & LOC_RS_CTRL);
                while (cm) {
                    const int g = (__ffs(cm) - 1) >> 3;
                    cm &= ~(0xffu << (8 * g));
                    const uint4 gh = lds128u(tb + L::OFF_REC + g * L::GSB + r * L::RECB + 16);
                    const unsigned gop = gh.z >> 24, gx = gh.x;
                    float *gs = sn_all + g * specs + row0;
                    float *slot = slots_warp + ((long long)g * P.nslot + gx) * spec + row0;
                    if (gop == LOC_OP_BG) {
                        for (int t = 0; t < O::NW; t++) {
                            const float bg = P.S.bgocc[P.slot0 + O::TB + t];
                            for (int c = 4 * lane; c < nchp; c += 128) *reinterpret_cast<float4 *>(gs + t * nchp + c) = make_float4(bg, bg, bg, bg);
                        }
                    } else if (gop == LOC_OP_SAVE) {
                        for (int i = lane * 4; i < rown; i += 128) stg_keep(slot + i, *reinterpret_cast<const float4 *>(gs + i), pol_keep);
                    } else if (gop == LOC_OP_LOAD) {
                        // all loads of a batch in flight before the first store: one L2 latency per batch, not per quad
                        constexpr int NB = 6;
                        for (int i0 = lane * 4; i0 < rown; i0 += 128 * NB) {
                            float4 v[NB];
#pragma unroll
                            for (int k = 0; k < NB; k++)
                                if (i0 + 128 * k < rown) v[k] = ldg_keep(slot + i0 + 128 * k, pol_keep);
#pragma unroll
                            for (int k = 0; k < NB; k++)
                                if (i0 + 128 * k < rown) *reinterpret_cast<float4 *>(gs + i0 + 128 * k) = v[k];
                        }
                    }
                }
                __syncwarp();
            }
            if (!(cls & LOC_RS_STEP)) continue;
            const float4 h0 = lds128(rb);
            const unsigned wbop = __float_as_uint(h0.w);
            const float4 qw = lds128(rb + L::QW);
            // photons emitted outside the updated channels escape (DESIGN 5.3): analytic mass of the wings for a common
            // round (qe >= 0), else the round sums the sampled profile itself: w (1 - sum phi), folded into b (fast_round)
            float qe = qw.z;
            if (cls & LOC_RS_SLOW) qe = -1.0f;
            else if (mode & LOC_RS_WIDE) qe = qew;
            const float fold = qe < 0.0f ? 1.0f : 0.0f;
            float2 ab[O::NHR * 2];
#pragma unroll
            for (int i = 0; i < O::NHR * 2; i++) ab[i] = make_float2(0.f, 0.f);
            if (__builtin_expect((cls & LOC_RS_SLOW) != 0, 0)) {
                hfsact += slow_round<NT, W, HFS>(P, rb, sq_g, pl, l8, nchp);
#pragma unroll
                for (int i = 0; i < O::NW; i++) ab[i] = lds64(pl + (O::TB + i) * L::ROWB);
            } else {
                // wing extension: the lane's channel among the LOC_EXT below / above the span, if inside the band (records that
                // are not steps have phi = 0 and all-zero coefficients)
                const int wb0 = (int)(wbop & LOC_WB_MASK);
                const int ce = wb0 + e0;
                const bool ext = ce >= 0 && ce < P.nch;
                const unsigned se = ext ? sq_r + 4u * ce : sq_g + 4u * wb0;
                const float pe = ext ? ex2f(fmaf(je, fmaf(je, h0.z, h0.y), h0.x)) : 0.0f;
                if (W != 2 || __builtin_expect(!(cls & LOC_RS_WIDE), 1)) {
                    fast_round<NT, W>(rb, sq_g + 4u * wb0, rowb, h0, J01, J23, se, pe, ext, fold, ab);
                } else {
                    // two passes: a WIDE ray over its pair of spans, the other rays over their span and then over nothing
                    const bool wide = mode & LOC_RS_WIDE;
                    const int w1 = wide ? wide_start(P.nch, lds32(rb + 28)) : wb0;
                    const float d1 = (float)(w1 - wb0), d2 = d1 + (float)LOC_SPAN;
                    float4 ha = h0, hb = h0;  // the profile's quadratic, re-centred on the spans that start at w1 and w1 + 32
                    ha.x = fmaf(d1, fmaf(d1, h0.z, h0.y), h0.x);
                    ha.y = fmaf(2.0f * d1, h0.z, h0.y);
                    hb.x = wide ? fmaf(d2, fmaf(d2, h0.z, h0.y), h0.x) : -INFINITY;
                    hb.y = fmaf(2.0f * d2, h0.z, h0.y);
                    // (a ray of the round that is not WIDE itself keeps its wing extension in the first pass)
                    fast_round<NT, W>(rb, sq_g + 4u * w1, rowb, ha, J01, J23, wide ? sq_g + 4u * w1 : se, wide ? 0.0f : pe, ext && !wide, fold, ab);
                    fast_round<NT, W>(rb, sq_g + 4u * (wide ? w1 + LOC_SPAN : w1), rowb, hb, J01, J23, sq_g + 4u * w1, 0.0f, false, fold, ab);
                }
            }
            // ---- reduction over the 8 lanes of each group in registers (halving butterfly: about 2 NW shuffles for the NW
            //      pairs): lane `own` ends up with the totals (A, B) of the warp's own-th transition and issues the two float
            //      atomics of (cell, transition) as one 64-bit RED ----
            float va[O::NHR * 2], vb[O::NHR * 2];
#pragma unroll
            for (int i = 0; i < O::NW; i++) {
                va[i] = ab[i].x;
                vb[i] = ab[i].y;
            }
            {
                int b0 = 0, n0 = O::NW, b1 = 0, n1 = O::NW;
                MultiReduce<O::NW, 4>::run(va, lane, b0, n0);
                MultiReduce<O::NW, 4>::run(vb, lane, b1, n1);
            }
            const bool step = wbop & LOC_RS_STEP;
            const uint4 h1 = lds128u(rb + 16);  // coff, w, opdz, cc
            if (step && own >= 0) {
                const float sc = lds32(rb + L::SC + 4 * (O::TB + own));
                const float w = __uint_as_float(h1.y);
                const float wesc = qe < 0.0f ? w : w * qe;
                float2 *cn = cnt_o + h1.x;
                asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(cn), "f"(va[0] * sc), "f"(fmaf(vb[0], sc, wesc)) : "memory");
            }
            if (O::HEAD && __builtin_expect(P.geom != 0, 0) && step && l8 == 0) {
                const unsigned cellidx = (h1.x - (unsigned)P.slot0) / (unsigned)P.nsp;
                atomicAdd(&P.visits[cellidx], 1u);
                atomicAdd(&P.pathz[cellidx], h1.z & 0x1fffffu);
            }
            __syncwarp();  // the next round's quads were written by other lanes
        }
        off += LOC_CHUNK;
        r0 = r1;
        r1 = r2;
    }
    if (O::HEAD) {  // per-warp totals
        unsigned long long ms = mysteps;
        for (int o = 16; o >= 1; o >>= 1) {
            ms += __shfl_xor_sync(0xffffffffu, ms, o);
            myactive += __shfl_xor_sync(0xffffffffu, myactive, o);
        }
        if (lane == 0 && ms) atomicAdd(P.nsteps, ms);
        // active updates = active channels of the steps x traced transitions (loc_stats.active_updates) ...
        if (P.geom && !HFS && lane == 0 && myactive) atomicAdd(P.nactive, myactive * (unsigned long long)P.nsel_all);
    }
    if (HFS && P.geomact) {  // ... with hyperfine structure counted transition by transition in the masked round (every warp its own)
        for (int o = 16; o >= 1; o >>= 1) hfsact += __shfl_xor_sync(0xffffffffu, hfsact, o);
        if (lane == 0 && hfsact) atomicAdd(P.nactive, hfsact);
    }
}

// The two-warp CTA runs two different instruction streams (each warp's transitions, the header work), and its time follows
// the size of the loop body (instruction-fetch stalls: profiles/r2_sim3d.md): the two-span WIDE round -- two more copies of
// the common round -- is compiled into the one-warp kernel only (C5: 580 vs 592 ms without it); in the two-warp kernel the
// few steps that need more than span + extension take the masked round instead (C3 57.7 -> 50.6 ms, C4 1012 -> 880 ms).
template <int NT, int NCHP_T, bool ONE, bool HFS>
__global__ void __maxnreg__(128) k_sim3d(Sim3D P)
{
    extern __shared__ __align__(16) float smem[];  // [4][NT][nchp] spectra, then the tables of Lay<NT>
    if (ONE)
        run_warp<NT, NCHP_T, 2, HFS>(P, smem);
    else if (threadIdx.x < 32)
        run_warp<NT, NCHP_T, 0, HFS>(P, smem);
    else
        run_warp<NT, NCHP_T, 1, HFS>(P, smem);
}

#define LOC_ONE_WARP_MAXNT 6  // one-warp CTAs are compiled up to this many transitions (the round keeps them all in registers)

template <int NT, int NCHP_T, bool ONE, bool HFS = false>
static int launch3d_t(loc_model *m, Sim3D &P, size_t smem)
{
    auto kern = k_sim3d<NT, NCHP_T, ONE, HFS>;
    const int nthr = ONE ? 32 : 64;
    LOC_CUDA_CHECK(m, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int bps = 0;
    LOC_CUDA_CHECK(m, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, nthr, smem));
    if (bps < 1) bps = 1;
    long long blocks = (long long)m->nsm * bps;
    blocks = std::min<long long>(blocks, (m->ntask + LOC_GROUPS - 1) / LOC_GROUPS);
    blocks = std::min<long long>(blocks, m->max_warps);
    if (blocks < 1) blocks = 1;
    LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_queue, 0, sizeof(unsigned int), m->stream));
    kern<<<(unsigned)blocks, nthr, smem, m->stream>>>(P);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    return LOC_OK;
}

static size_t spectra_bytes(int nt, int nchp) { return sizeof(float) * LOC_GROUPS * ((size_t)nt * nchp + LOC_RAY_SKEW); }

template <int NT>
static int launch3d(loc_model *m, Sim3D &P)
{
    const size_t smem = spectra_bytes(NT, P.nchp) + Lay<NT>::BYTES;
    if (smem > 200 * 1024 || P.nch > (int)LOC_WB_MASK || P.nch > 0xffff) {
        snprintf(m->err, sizeof(m->err), "nchannel * ntrans too large for the shared-memory spectra (%zu bytes per warp)", smem);
        return LOC_EINVAL;
    }
    if (P.H.any) return launch3d_t<NT, 0, false, true>(m, P, smem);  // hyperfine structure: every step takes the masked round
    // one warp per ray set for few transitions (loc_set_option(LOC_OPT_SIM3D_WARPS): 0 = automatic: up to 4 transitions)
    if constexpr (NT <= LOC_ONE_WARP_MAXNT) {
        if (m->sim3d_warps == 1 || (m->sim3d_warps == 0 && NT <= 4)) {
            if (P.nchp == 128) return launch3d_t<NT, 128, true>(m, P, smem);
            if (P.nchp == 256) return launch3d_t<NT, 256, true>(m, P, smem);
            return launch3d_t<NT, 0, true>(m, P, smem);
        }
    }
    if (P.nchp == 128) return launch3d_t<NT, 128, false>(m, P, smem);
    if (P.nchp == 256) return launch3d_t<NT, 256, false>(m, P, smem);
    return launch3d_t<NT, 0, false>(m, P, smem);
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
    P.xclip = m->xclip;
    P.xfull = m->xfull;
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
    P.nactive = m->d_steps + 1;
    P.queue = m->d_queue;
    P.pool = m->spec_pool;
    P.S = m->selh;
    P.nsel_all = m->selh.nsel;
    loc_fill_hfs(m, P.H);
    if ((long long)m->ncell * P.nsp >= (1ll << 32)) {
        snprintf(m->err, sizeof(m->err), "ncell * ntrans exceeds the 32-bit counter offsets of the 3D kernel");
        return LOC_EINVAL;
    }
    // All traced transitions go through one launch while the spectra of a warp's four rays fit 24 KB of shared memory
    // (9 transitions x 128 channels = 18 KB); otherwise they are split into `npart` launches of nearly equal size, at the
    // price of repeating the per-step work (profiles/r1_v5_sim3d_C3.md: ~10 ms per extra launch on C3).
    int nsel = m->selh.nsel;
    int npart = 1;
    while (npart < nsel && spectra_bytes((nsel + npart - 1) / npart, P.nchp) > 24 * 1024) npart++;
    if (m->sim3d_parts > 0) npart = std::max(npart, std::min(nsel, m->sim3d_parts));  // loc_set_option(LOC_OPT_SIM3D_PARTS)
    int slot = 0;
    for (int part = 0; part < npart; part++) {
        int n = (nsel - slot + (npart - part) - 1) / (npart - part);
        if (part + 1 < npart) n = std::min(nsel - slot, (n + 1) & ~1);  // even parts: 16-byte aligned coefficient records
        P.slot0 = slot;
        int rc = LOC_EINVAL;
        // the step / active-channel statistics are taken by the first part only
        P.geom = geom && part == 0;
        P.geomact = geom && (part == 0 || P.H.any);
        unsigned long long *keep = P.nsteps;
        if (part > 0) P.nsteps = m->d_steps + 2;  // scratch slot
        switch (n) {
#define C3(N)                     \
    case N:                       \
        rc = launch3d<N>(m, P);   \
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
