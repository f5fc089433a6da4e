// loc_paths3d.cu -- 3D octree / Cartesian ray paths: the set-up half of the 3D ray tracing.
//
// Two parts (the second lives in loc_sim3d.cu):
//  (1) PATH BUILDER (set-up, runs when the directions are set): one thread per root-grid ray.  It walks the ray and
//      every ray born from it in refined regions through the octree with INTEGER arithmetic only
//      (DESIGN R7) and writes the result as a linear "step stream" of 8-byte records: STEP(cell, dzeta) plus the three
//      spectrum operations BG / SAVE(slot) / LOAD(slot) that encode births, wrap-arounds and the return to the parent
//      ray.  The paths depend only on the grid and the directions, not on the level populations, so -- like the
//      per-shell path lengths of the 1D model that the paper pre-calculates -- they are computed once
//      and kept in HBM (B200: 180 GB) instead of being recomputed by one idle-lane-surrounded work item per step
//      (the paper's stated bottleneck).
//  (2) RADIATIVE KERNEL (every ALI iteration): a quarter-warp per root-ray task, four tasks per CTA of one or two warps
//      (loc_sim3d.cu), lanes over the velocity channels of the local profile window.  It streams the records, evaluates the Doppler-shifted profile, optical depths, Eq. 3 and
//      the two per-cell sums (Eq. 2 first term and the escape fraction) for all traced transitions at once.
#include <stdio.h>

#include <algorithm>
#include <vector>

#include "loc_internal.cuh"

// ------------------------------------------------------------------------------------------------
// direction set-up (host)
// ------------------------------------------------------------------------------------------------
void loc_fill_dir(loc_model *m, const double *din, Dir3 *D)
{
    int n[3] = {m->nx, m->ny, m->nz};
    int mm = 0;
    for (int a = 1; a < 3; a++)
        if (fabs(din[a]) > fabs(din[mm])) mm = a;  // ties -> lowest axis index
    D->ax[0] = mm;
    D->ax[1] = (mm + 1) % 3;
    D->ax[2] = (mm + 2) % 3;
    double sl[2];
    for (int k = 0; k < 2; k++) {
        double s = fabs(din[D->ax[k + 1]]) / fabs(din[mm]);
        unsigned long long S = (unsigned long long)nearbyint(s * (double)LOC_H0);  // round half even (DESIGN R7)
        if (S == 0) {
            D->T[k] = 0;
            D->M[k] = 0;
            sl[k] = 0.0;
        } else {
            D->T[k] = ((1ull << 52) + S / 2) / S;
            D->M[k] = (unsigned long long)((((unsigned __int128)1) << 64) / D->T[k]);
            sl[k] = 4294967296.0 / (double)D->T[k];
        }
    }
    double lenf = sqrt(1.0 + sl[0] * sl[0] + sl[1] * sl[1]);
    for (int k = 0; k < 3; k++) {
        D->flip[k] = din[D->ax[k]] < 0.0;
        D->W[k] = n[D->ax[k]] * LOC_H0;
    }
    D->d[D->ax[0]] = (float)((D->flip[0] ? -1.0 : 1.0) / lenf);
    D->d[D->ax[1]] = (float)((D->flip[1] ? -1.0 : 1.0) * sl[0] / lenf);
    D->d[D->ax[2]] = (float)((D->flip[2] ? -1.0 : 1.0) * sl[1] / lenf);
    D->sf = (float)(m->root_cm / (double)LOC_H0 * lenf);
    D->np = n[D->ax[1]];
    D->nq = n[D->ax[2]];
    D->task0 = 0;
}

struct Pending {  // 16 bytes
    int bp, bq, zeta;
    unsigned char tag, src, resumed, pad;  // src: slot index, or 255 = background
};
#define LOC_SRC_BG 255

struct BuildArgs {
    Tree G;
    const Dir3 *dirs;
    const uint16_t *task_dir;
    long long task_begin, task_end;
    long long *task_off;  // count pass: counts written to task_off[task]; emit pass: offsets read from it
    uint2 *stream;
    Pending *stacks;
    int *errflag;
    unsigned long long *nsteps;
    int emit;
};

// Path builder: traces root line `task` and all its descendants depth first (DESIGN 6.3).
// SIMT shape.  A thread's sequence of operations is the plain depth-first walk; what the warp executes is arranged in two
// phases per round so that the long, rare part does not serialise the short, common one: phase 1 -- every lane steps its
// ray from leaf to leaf until the ray ends or stands on the upstream face of a refined ancestor (a possible donor event);
// phase 2 -- after the warp has reconverged, the lanes that stopped for a donor event evaluate it together (the same 21
// candidate positions each), then step.  Taken lane by lane inside one loop, the donor evaluation (~1300 instructions even
// when it finds nothing) was paid by the whole warp in 9 of 10 iterations (C4: 6.9 s of set-up).
// steps a lane may take in phase 1 before the warp looks at the donor events collected so far (C4 set-up: unlimited 2.74 s,
// 24 -> 2.48 s, 8 -> 2.28 s: lanes that stopped early do not wait for the longest event-free run of the warp)
#define LOC_BUILD_K 8
__global__ void __launch_bounds__(128) k_build_paths(BuildArgs A)
{
    const long long task = A.task_begin + blockIdx.x * (long long)blockDim.x + threadIdx.x;
    bool finished = task >= A.task_end;  // such lanes stay for the warp-wide votes
    const Tree &G = A.G;
    const Dir3 D = A.dirs[finished ? 0 : A.task_dir[task]];
    Pending *stack = A.stacks + (blockIdx.x * (long long)blockDim.x + threadIdx.x) * LOC_BUILD_STACK;
    int sp = 0;
    long long nrec = 0, nstep = 0;
    uint2 *out = (A.emit && !finished) ? A.stream + A.task_off[task] : nullptr;
    const int Wz = D.W[0], Wp = D.W[1], Wq = D.W[2];
    if (!finished) {
        long long lt = task - D.task0;
        const int O_p = 25 * (LOC_H0 / 64), O_q = 41 * (LOC_H0 / 64);  // DESIGN R8
        Pending r;
        r.bp = O_p + (int)(lt % D.np) * LOC_H0;
        r.bq = O_q + (int)(lt / D.np) * LOC_H0;
        r.zeta = 0;
        r.tag = 0;
        r.src = LOC_SRC_BG;
        r.resumed = 0;
        r.pad = 0;
        stack[sp++] = r;
    }
#define EMIT(x_, y_)                             \
    do {                                         \
        if (out) out[nrec] = make_uint2(x_, y_); \
        nrec++;                                  \
    } while (0)
    // step through the leaf L from zeta
#define STEP_LEAF()                                                                                              \
    do {                                                                                                         \
        const int h = LOC_H0 >> L.level;                                                                         \
        long long znext = (zeta & ~(long long)(h - 1)) + h, z;                                                   \
        z = cross_of(D.T[0], Sp + (fp & ~(h - 1)) + h - fp); if (z < znext) znext = z;                           \
        z = cross_of(D.T[1], Sq + (fq & ~(h - 1)) + h - fq); if (z < znext) znext = z;                           \
        EMIT((unsigned)L.cell[L.level], LOC_REC(LOC_OP_STEP, L.level, (unsigned)(znext - zeta)));                \
        nstep++;                                                                                                 \
        zeta = znext;                                                                                            \
        first = false;                                                                                           \
    } while (0)
    int just_saved = -1;  // slot of the SAVE that was the last record emitted (-1: the last record was something else)
    // state of the ray being walked
    Pending cur;
    cur.bp = cur.bq = cur.zeta = 0;
    cur.tag = cur.src = cur.resumed = cur.pad = 0;
    int tag = 0, fp = 0, fq = 0;
    long long zeta = 0, wrp = 0, wrq = 0, Sp = 0, Sq = 0;
    bool first = true, walking = false;
    LeafPos L;
    L.level = 0;
    for (;;) {
        if (__all_sync(0xffffffffu, finished)) break;
        // ---- next ray of this root line ----
        if (!finished && !walking) {
            if (sp == 0) {
                while (nrec & (LOC_TASK_ALIGN - 1)) EMIT(0u, LOC_REC(LOC_OP_NOP, 0, 0));  // tasks are whole chunks of records
                if (!A.emit) {
                    A.task_off[task] = nrec;
                    atomicAdd(A.nsteps, (unsigned long long)nstep);
                }
                finished = true;
            } else {
                cur = stack[--sp];
                tag = cur.tag;
                // the ray starts from the background or from a saved spectrum; the first ray served after a SAVE finds that
                // very spectrum still in place, so its LOAD is left out (a quarter of all LOADs of a refined model)
                if (cur.src == LOC_SRC_BG)
                    EMIT(0u, LOC_REC(LOC_OP_BG, 0, 0));
                else if ((int)cur.src != just_saved)
                    EMIT((unsigned)cur.src, LOC_REC(LOC_OP_LOAD, 0, 0));
                just_saved = -1;
                zeta = cur.zeta;
                first = true;
                wrp = wrq = 0;
                walking = true;
            }
        }
        // ---- phase 1: leaf to leaf until the ray ends or may have donor duty ----
        bool donor = false;
        if (!finished) {
            int budget = LOC_BUILD_K;
            while (walking && budget-- > 0) {
                if (zeta >= Wz) {
                    walking = false;
                    break;
                }
                Sp = shift_of(D, 0, zeta);
                Sq = shift_of(D, 1, zeta);
                const long long up = cur.bp + Sp, uq = cur.bq + Sq;
                long long rp, rq;
                const long long wp_ = wrap_of(up, Wp, rp), wq_ = wrap_of(uq, Wq, rq);
                fp = (int)rp;
                fq = (int)rq;
                const bool wrapped = !first && (wp_ != wrp || wq_ != wrq);
                wrp = wp_;
                wrq = wq_;
                find_leaf(G, D, (int)zeta, fp, fq, L);
                if (L.level < tag) {  // entering a region refined to less than the tag: terminated
                    walking = false;
                    break;
                }
                if (wrapped) EMIT(0u, LOC_REC(LOC_OP_BG, 0, 0));  // left through a side, re-enters opposite
                // donor duty is possible where the ray stands on the upstream face of a refined ancestor
                if (!(first && cur.resumed))
                    for (int j = tag; j < L.level; j++) donor |= !(zeta & ((LOC_H0 >> j) - 1));
                if (donor) break;
                STEP_LEAF();
            }
        }
        __syncwarp();
        // ---- phase 2: donor duty: upstream face of refined ancestors entered now ----
        if (donor) {
            int saved = -1;
            for (int j = tag; j < L.level; j++) {
                const int hj = LOC_H0 >> j, hk = hj >> 1;
                if (zeta & (hj - 1)) continue;
                const int op = fp & ~(hj - 1), oq = fq & ~(hj - 1);
                for (int dj = -3; dj <= 1; dj++)
                    for (int di = -3; di <= 1; di++) {
                        if (!((di | dj) & 1)) continue;  // member of the coarser lattice P_j
                        const long long ap = (long long)fp + di * hk, aq = (long long)fq + dj * hk;
                        long long zin = zeta, zout = zeta + hj, z;
                        z = cross_of(D.T[0], Sp + op - ap); if (z > zin) zin = z;
                        z = cross_of(D.T[1], Sq + oq - aq); if (z > zin) zin = z;
                        z = cross_of(D.T[0], Sp + op + hj - ap); if (z < zout) zout = z;
                        z = cross_of(D.T[1], Sq + oq + hj - aq); if (z < zout) zout = z;
                        if (zout <= zin) continue;  // does not cross this cell
                        int src = -1;               // -1: slot of this event
                        if (zin == 0) {
                            src = LOC_SRC_BG;
                        } else {
                            const long long zb = zin - 1;
                            const long long pb = ap + shift_of(D, 0, zb) - Sp, qb = aq + shift_of(D, 1, zb) - Sq;
                            const long long pi = ap + shift_of(D, 0, zin) - Sp, qi = aq + shift_of(D, 1, zin) - Sq;
                            long long rpb, rqb, rdummy;
                            const long long wpb = wrap_of(pb, Wp, rpb), wqb = wrap_of(qb, Wq, rqb);
                            if (level_at(G, D, (int)zb, (int)rpb, (int)rqb) >= j + 1) continue;  // alive already
                            if (wpb != wrap_of(pi, Wp, rdummy) || wqb != wrap_of(qi, Wq, rdummy)) src = LOC_SRC_BG;
                        }
                        if (saved < 0) {
                            saved = j;
                            just_saved = j;
                            EMIT((unsigned)j, LOC_REC(LOC_OP_SAVE, 0, 0));
                            if (sp < LOC_BUILD_STACK) {
                                Pending c = cur;
                                c.zeta = (int)zeta;
                                c.src = (unsigned char)j;
                                c.resumed = 1;
                                stack[sp++] = c;
                            } else
                                *A.errflag = 1;
                        }
                        if (sp < LOC_BUILD_STACK) {
                            Pending c;
                            long long bb, bc;
                            wrap_of(ap - Sp, Wp, bb);
                            wrap_of(aq - Sq, Wq, bc);
                            c.bp = (int)bb;
                            c.bq = (int)bc;
                            c.zeta = (int)zin;
                            c.tag = (unsigned char)(j + 1);
                            c.src = (unsigned char)(src == LOC_SRC_BG ? LOC_SRC_BG : saved);
                            c.resumed = 0;
                            c.pad = 0;
                            stack[sp++] = c;
                        } else
                            *A.errflag = 1;
                    }
            }
            if (saved >= 0)
                walking = false;  // children first; this ray resumes from the saved spectrum afterwards
            else
                STEP_LEAF();
        }
    }
#undef STEP_LEAF
#undef EMIT
}

// exclusive scan of counts[0..n) in place (one block), total written to counts[n]
__global__ void __launch_bounds__(1024) k_scan_tasks(long long *counts, long long n)
{
    __shared__ long long part[1024];
    const int tid = threadIdx.x;
    const long long per = (n + 1023) / 1024;
    const long long b = tid * per, e = (b + per < n) ? b + per : n;
    long long s = 0;
    for (long long i = b; i < e; i++) s += counts[i];
    part[tid] = s;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
        long long v = (tid >= o) ? part[tid - o] : 0;
        __syncthreads();
        part[tid] += v;
        __syncthreads();
    }
    long long run = part[tid] - s;
    for (long long i = b; i < e; i++) {
        long long c = counts[i];
        counts[i] = run;
        run += c;
    }
    if (tid == 1023) counts[n] = part[1023];
}

__global__ void k_check_tree(Tree G, int *errflag)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = G.noff[G.nlev];
    if (i >= n) return;
    int l = 0;
    while (i >= G.noff[l + 1]) l++;
    int ch = G.child[i];
    if (ch < 0) return;
    if (l + 1 >= G.nlev || (ch & 7) || (long long)ch + 8 > G.noff[l + 2] - G.noff[l + 1]) *errflag = 2;
}

int loc_setup3d(loc_model *m)
{
    Tree G = make_tree(m);
    LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_errflag, 0, sizeof(int), m->stream));
    int64_t n = m->ncell;
    k_check_tree<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(G, m->d_errflag);
    m->launches++;
    LOC_CUDA_CHECK(m, cudaGetLastError());
    int err = 0;
    LOC_CUDA_CHECK(m, cudaMemcpyAsync(&err, m->d_errflag, sizeof(int), cudaMemcpyDeviceToHost, m->stream));
    LOC_CUDA_CHECK(m, cudaStreamSynchronize(m->stream));
    if (err) {
        snprintf(m->err, sizeof(m->err), "octree child index out of range or not a multiple of 8");
        return LOC_EINVAL;
    }
    return LOC_OK;
}

// Builds the step stream of `ndir` directions (already in m->h_dirs / m->d_dirs) with `ntask` root-line tasks.  Commits
// m->stream_len / setup_steps / setup_ms only on success; the caller commits m->ndir / m->ntask.
static int build_streams_timed(loc_model *m, int ndir, int64_t ntask, cudaEvent_t e0, cudaEvent_t e1)
{
    LOC_CUDA_CHECK(m, cudaEventRecord(e0, m->stream));
    // task -> direction table
    {
        std::vector<uint16_t> td((size_t)ntask);
        for (int i = 0; i < ndir; i++) {
            int64_t n = (int64_t)m->h_dirs[i].np * m->h_dirs[i].nq;
            std::fill(td.begin() + m->h_dirs[i].task0, td.begin() + m->h_dirs[i].task0 + n, (uint16_t)i);
        }
        LOC_CUDA_CHECK(m, cudaMemcpyAsync(m->d_task_dir, td.data(), td.size() * sizeof(uint16_t), cudaMemcpyHostToDevice, m->stream));
        LOC_CUDA_CHECK(m, cudaStreamSynchronize(m->stream));
    }
    BuildArgs A;
    A.G = make_tree(m);
    A.dirs = m->d_dirs;
    A.task_dir = m->d_task_dir;
    A.task_off = m->d_task_off;
    A.stream = m->d_stream;
    A.stacks = (Pending *)m->d_bstack;
    A.errflag = m->d_errflag;
    A.nsteps = m->d_steps;
    LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_errflag, 0, sizeof(int), m->stream));
    LOC_CUDA_CHECK(m, cudaMemsetAsync(m->d_steps, 0, sizeof(unsigned long long), m->stream));
    long long total = 0;
    unsigned long long steps = 0;
    for (int pass = 0; pass < 2; pass++) {
        A.emit = pass;
        for (int64_t b = 0; b < ntask; b += m->bstack_threads) {
            A.task_begin = b;
            A.task_end = std::min<int64_t>(ntask, b + m->bstack_threads);
            unsigned nb = (unsigned)((A.task_end - A.task_begin + 127) / 128);
            k_build_paths<<<nb, 128, 0, m->stream>>>(A);
            m->launches++;
            LOC_CUDA_CHECK(m, cudaGetLastError());
        }
        if (pass == 0) {
            k_scan_tasks<<<1, 1024, 0, m->stream>>>(m->d_task_off, ntask);
            m->launches++;
            LOC_CUDA_CHECK(m, cudaGetLastError());
            int err = 0;
            LOC_CUDA_CHECK(m, cudaMemcpyAsync(&total, m->d_task_off + ntask, sizeof(total), cudaMemcpyDeviceToHost, m->stream));
            LOC_CUDA_CHECK(m, cudaMemcpyAsync(&steps, m->d_steps, sizeof(steps), cudaMemcpyDeviceToHost, m->stream));
            LOC_CUDA_CHECK(m, cudaMemcpyAsync(&err, m->d_errflag, sizeof(err), cudaMemcpyDeviceToHost, m->stream));
            LOC_CUDA_CHECK(m, cudaStreamSynchronize(m->stream));
            if (err) {
                snprintf(m->err, sizeof(m->err), "path builder: more than %d pending rays on one root ray", LOC_BUILD_STACK);
                return LOC_ENOMEM;
            }
            if (total > m->stream_cap) {
                // the message carries the required record count: the workspace is sized for 3 ncell ndir_max + 16 ntask_max
                // records (loc_workspace_bytes); a caller that hits this creates the model with a larger ndir_max
                snprintf(m->err, sizeof(m->err), "step stream needs %lld records (8 bytes each), workspace holds %lld: create the model with a larger ndir_max",
                         total, (long long)m->stream_cap);
                return LOC_ENOMEM;
            }
        }
    }
    LOC_CUDA_CHECK(m, cudaEventRecord(e1, m->stream));
    LOC_CUDA_CHECK(m, cudaEventSynchronize(e1));
    float ms = 0.f;
    LOC_CUDA_CHECK(m, cudaEventElapsedTime(&ms, e0, e1));
    m->stream_len = total;
    m->setup_steps = (int64_t)steps;
    m->setup_ms = ms;
    return LOC_OK;
}

int loc_build_streams(loc_model *m, int ndir, int64_t ntask)
{
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        if (e0) cudaEventDestroy(e0);
        snprintf(m->err, sizeof(m->err), "cudaEventCreate failed");
        return LOC_ECUDA;
    }
    const int rc = build_streams_timed(m, ndir, ntask, e0, e1);  // the events are destroyed on every exit path
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return rc;
}
