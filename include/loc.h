/*
 * loc.h -- C-ABI boundary of the B200-native LOC hot path (arxiv 2009.12609, M. Juvela).
 *
 * The library runs the ray-tracing simulation step of accelerated lambda iteration (ALI) and the
 * per-cell statistical-equilibrium solve on one GPU (hand-written CUDA for sm_100a).  Citations are
 * PAPER.md:<line> of /root/reference/PAPER.md; "DESIGN Rn" are the readings listed in DESIGN.md.
 *
 * Conventions
 *   - Units are CGS everywhere (cm, cm/s, K, cm^-3, 1/s).
 *   - Every call returns an int status: LOC_OK or a negative LOC_E* code.  No exceptions, no exit().
 *     loc_last_error() returns a static/owned message for the last failing call on that model.
 *   - "host" pointers are ordinary CPU memory, read during the call only (the library copies what it
 *     needs).  "device" pointers are CUDA global memory of the current device, OWNED BY THE CALLER and
 *     kept alive by the caller until loc_destroy_model().
 *   - The library performs NO hidden device allocation: all device scratch lives in the caller's
 *     workspace (loc_workspace_bytes / loc_create_model).  Too small a workspace -> LOC_ENOMEM.
 *   - All device work is enqueued on the stream given to loc_create_model and is asynchronous; only calls
 *     that return a host scalar (loc_solve, loc_iterate, loc_get_stats) synchronise that stream.
 *   - Channel c of NCH has velocity v_c = (c - (NCH-1)/2) dv, dv = 2 band_halfwidth / NCH (DESIGN O4).
 *   - Doppler shift of a cell with velocity v seen along the photon direction d is v0 = -(v . d)
 *     (radio convention, DESIGN R6); in 1D v0 = -v_r mu with mu evaluated where the ray ENTERS the step
 *     ("the Doppler shifts are evaluated only at the beginning of each step").
 */
#ifndef LOC_H
#define LOC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LOC_OK 0
#define LOC_EINVAL (-1) /* bad argument (non-monotone radii, nchannel<1, child index out of range, ...) */
#define LOC_ESTATE (-2) /* call order (species / directions / populations not set)                      */
#define LOC_ENOMEM (-3) /* workspace too small                                                          */
#define LOC_ECUDA (-4)  /* CUDA error; text in loc_last_error()                                        */
#define LOC_ENONFINITE (-5) /* loc_solve / loc_iterate* produced a NaN or infinite population (T_kin <= 0, NaN inputs):
                               max_rel_change is +inf; never reported as "converged"                      */

#define LOC_GRID_SHELL 1  /* 1D spherically symmetric shells   */
#define LOC_GRID_OCTREE 2 /* 3D octree; a Cartesian grid is nlevel = 1 */

#define LOC_MAX_TRANS 12  /* radiative transitions ray traced together in one pass */
#define LOC_MAX_LEVELS 32 /* energy levels of the species                           */
#define LOC_MAX_TREE_LEVELS 6
#define LOC_MAX_DIRECTIONS 65535 /* ray directions of one model (loc_set_directions)                    */
#define LOC_MAX_HFS 8            /* hyperfine components of one transition (loc_set_hyperfine)          */

/* Keys of loc_set_option.  The library reads NO environment variables: every knob that can change a result or a launch
 * configuration is an argument of this call (defaults in parentheses; DESIGN.md 5.3 derives them).                    */
#define LOC_OPT_WINDOW_XMIN 1    /* (4.5) 1D kernel and the masked path of the 3D kernel: channels within X sigma of the line
                                    centre are updated, X^2 = xmin^2 + 2 ln max(1, dv/sigma)^2 (+ the optical-depth term)  */
#define LOC_OPT_WINDOW_EPS_TAU 2 /* (1e-6) 1D kernel: X >= sqrt(2 ln(tau0 / eps_tau)), tau0 = largest line-centre optical
                                    depth of the step                                                                     */
#define LOC_OPT_SPAN_XCLIP 3     /* (3.4) 3D kernel: a step whose 32-channel span does not reach X sigma, X^2 = xclip^2 +
                                    2 ln max(1, tau0), takes two spans or the masked path (beyond X sigma the optical depth of
                                    the step is < 3e-3: the 8 channels below and above the span are carried to first order)  */
#define LOC_OPT_SPAN_XFULL 7     /* (4.8) 3D kernel: ... and the span with those 8 + 8 channels must reach X_f sigma, X_f^2 =
                                    xfull^2 + 2 ln max(1, tau0): what lies beyond is dropped (optical depth < 1e-5)          */
#define LOC_OPT_SIM3D_PARTS 4    /* (0 = automatic) 3D kernel: split the traced transitions over at least this many launches */
#define LOC_OPT_SOLVER 5         /* (0 = automatic: float32 in registers for species of <= 12 levels whose transitions and
                                    collisional pairs all run from the higher to the lower level index, else float64)
                                    1 = float64 solver with the matrix in local memory, 2 = float64 solver with the matrix in
                                    shared memory (<= 16 levels): A/B measurements and reference runs                    */
#define LOC_OPT_SOLVER_LOCAL LOC_OPT_SOLVER /* earlier name of the key */
#define LOC_OPT_SIM3D_WARPS 6    /* (0 = automatic: one warp per set of four rays up to 4 traced transitions per launch, else two
                                    warps that split the transitions) 1 = one warp where compiled (<= 6 transitions), 2 = two */

typedef struct loc_model loc_model; /* opaque */

/* Geometry (PAPER.md:87 for shells, PAPER.md:93-97 for the octree; storage format DESIGN R17). */
typedef struct {
    int kind; /* LOC_GRID_SHELL or LOC_GRID_OCTREE */
    /* --- shell grid: shell k spans [r_out[k-1], r_out[k]), r_out[-1] = 0; values refer to the shell */
    int nshell;
    const double *r_out; /* host [nshell], strictly ascending, cm                                         */
    int nray;
    const double *ray_p; /* host [nray] impact parameters, 0 <= p < r_out[nshell-1]                       */
    const double *ray_w; /* host [nray] ray weights = annulus areas pi (p_hi^2 - p_lo^2), cm^2 (Eq. 1)   */
    /* --- octree grid: level-major cell arrays; level l holds level_offset[l+1]-level_offset[l] cells.
     *     Root level in x-fastest raster order (ix + nx (iy + ny iz)); the 8 children of a refined cell are
     *     contiguous in the next level in (x fastest, y, z) order.                                          */
    int nx, ny, nz;              /* root grid dimensions                                                  */
    double root_cell_cm;         /* edge of a root cell                                                   */
    int nlevel;                  /* number of hierarchy levels >= 1 (<= LOC_MAX_TREE_LEVELS)              */
    const int64_t *level_offset; /* host [nlevel+1]; level_offset[nlevel] = total number of cells         */
    const int32_t *child;        /* DEVICE [ncell]: index WITHIN the next level of the first child, or -1 for a leaf */
} loc_grid;

/* Per-cell physical state, DEVICE float arrays over all cells (octree: leaves and refined
 * cells alike, in the level-major order of loc_grid; values of refined cells are ignored). */
typedef struct {
    const float *density;   /* number density of the collision partner, cm^-3                             */
    const float *tkin;      /* kinetic temperature, K                                                     */
    const float *sigma;     /* turbulent 1-D velocity dispersion (std dev), cm/s; thermal part added by the
                               library as k T / m unless species mass is 0 (DESIGN R3)                     */
    const float *vx;        /* velocity, cm/s; shells: radial velocity (positive outward)                 */
    const float *vy;        /* octree only                                                                */
    const float *vz;        /* octree only                                                                */
    const float *abundance; /* fractional abundance of the species relative to `density`                  */
} loc_cells;

typedef struct {
    int64_t ncell;           /* cells in the model (all levels)                                           */
    int64_t steps;           /* ray-cell steps of the last loc_simulate (one count per ray segment in a cell) */
    int ntrans_sim;          /* transitions traced in the last loc_simulate                               */
    int nchannel;
    int64_t kernel_launches; /* CUDA kernels launched by the library on this model so far                  */
    int counter_stride;      /* floats per cell in the counter / coefficient records = 2 * ntrans_padded  */
    int64_t active_channels; /* sum over the steps of the last loc_simulate(geometry_counters=1) of the number of
                                channels with |v_c - v_0| <= 5 sigma: the counting definition of "active" ray-cell-
                                channel updates per traced transition (DESIGN 8), independent of the kernel's window */
    int64_t setup_steps;     /* octree: ray-cell steps in the precomputed step stream (all directions)      */
    double setup_ms;         /* octree: device time of the last path set-up (loc_set_directions), ms        */
    int64_t active_updates;  /* the same count summed over the traced transitions: = active_channels x ntrans_sim without
                                hyperfine structure; with it a transition's active channels are those within 5 sigma of
                                any of its components, and active_channels = active_updates / ntrans_sim               */
} loc_stats;

/* Bytes of device workspace loc_create_model needs for this grid and these limits.
 * ndir_max: largest number of directions that will be set (octree; ignored for shells). */
int64_t loc_workspace_bytes(const loc_grid *grid, int nchannel, int nlevel_species, int ntrans, int ndir_max);

/* Build a model: validates the grid, precomputes the set-up tables (1D: per-ray path lengths, entry
 * cosines, sampled shell volumes V_eff = sum_i W_i s_ik, DESIGN R12; 3D: neighbour-refinement flags) in the
 * workspace.  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 * nchannel >= 1; band_halfwidth_cm_s > 0; t_background_K >= 0 (Planck background, Eq. 1).
 * nlevel_species, ntrans, ndir_max: the same limits that were given to loc_workspace_bytes; later calls to
 * loc_set_species / loc_set_directions must stay within them.                                          */
int loc_create_model(const loc_grid *grid, const loc_cells *cells, int nchannel, double band_halfwidth_cm_s,
                     double t_background_K, int nlevel_species, int ntrans, int ndir_max, void *workspace /* device */,
                     int64_t workspace_bytes, void *stream, loc_model **out);

/* Species: host arrays, copied.  Line frequencies follow from the level energies.  Upward
 * collision rates by detailed balance; rate_down is [ntemp][ncoll], linear interpolation in T, clamped;
 * ntemp = 1 -> constant.  mass_amu = 0 -> `sigma` is the total line width.  ntrans <= LOC_MAX_TRANS.     */
int loc_set_species(loc_model *m, int nlevel, const double *energy_K, const double *g, int ntrans, const int *upper,
                    const int *lower, const double *einstein_A, double mass_amu, int ncoll, const int *cu, const int *cl,
                    int ntemp, const double *temps_K, const double *rate_down);

/* Hyperfine structure with LTE between the components ("in the case of hyperfine spectra, assuming LTE
 * distribution between the hyperfine components"; PAPER.md:149 NH3(1,1), PAPER.md:388 HCN J = 1-0): transition `trans`
 * of the species consists of ncomp components; component k is a Gaussian of the cell's line width centred dv_cm_s[k] away
 * from the line centre on the channel velocity axis (positive = higher channel velocity) and carries the fraction
 * weight[k] of the line (weights > 0, sum 1 within 1e-6).  The levels keep ONE population each, so the components share
 * the source function; profile, optical depth and both counters of the transition use
 *     phi_c = sum_k weight[k] dv / (sigma sqrt(2 pi)) exp(-(v_c - v_0 - dv_cm_s[k])^2 / (2 sigma^2)).
 * Host arrays, copied.  ncomp = 0 (or 1 with zero offset) removes the structure; ncomp <= LOC_MAX_HFS.  Call after
 * loc_set_species (which clears all hyperfine structure).  Steps of a model with any hyperfine transition take the
 * kernels' general (masked-window) path.                                                                          */
int loc_set_hyperfine(loc_model *m, int trans, int ncomp, const double *dv_cm_s, const double *weight);

/* Re-read the caller's cell arrays (same device pointers as given to loc_create_model) after their content has been
 * changed from outside, and rebuild the derived per-cell kinematics record (velocity, total line width).     */
int loc_refresh_cells(loc_model *m);

/* Octree only: ray directions (unit vectors, host [ndir][3]; PAPER.md:93 uses HEALPix centres).  Each is
 * snapped to the library's fixed-point slopes (DESIGN R7); ndir <= the ndir_max given to loc_workspace_bytes
 * (<= LOC_MAX_DIRECTIONS).  On failure (LOC_ENOMEM: the message names the number of 8-byte records the step stream
 * needs; LOC_ECUDA) the model is left WITHOUT directions and loc_simulate returns LOC_ESTATE until a later call succeeds.
 * This call also runs the path set-up: every root-grid ray and the rays born from it in refined regions
 * are traced once with integer arithmetic and stored in the workspace as a step stream
 * (cell index, path length) that loc_simulate replays every iteration -- the 3D counterpart of the pre-calculated
 * per-shell path lengths of PAPER.md:87.  Synchronises the stream.  LOC_ENOMEM if the stream does not fit.      */
int loc_set_directions(loc_model *m, int ndir, const double *dir_xyz);

/* Register the caller-owned DEVICE population buffer, float [nlevel][ncell] (cm^-3), and derive the per-cell
 * line coefficients from its current content.  Call again after writing into the buffer from outside.    */
int loc_set_populations(loc_model *m, float *dev_pops);

/* Fill the registered buffer with LTE populations at T_kin and derive the coefficients.   */
int loc_init_lte(loc_model *m);

/* Zero the counters and trace all rays (1D: all impact parameters; 3D: all directions, root rays and the
 * rays born in refined regions) for the selected transitions (nsel = 0 -> all), evaluating
 * per cell step and channel the Doppler-shifted Gaussian profile, the optical depth, the photon
 * transfer of Eq. 3 and the sums of Eq. 2 (first term; the self term is handled by ALI).
 * The selection is remembered for loc_solve / loc_iterate.  geometry_counters != 0 additionally records
 * per-cell visit counts and integer main-axis path sums (tests).                                           */
int loc_simulate(loc_model *m, int nsel, const int *trans_idx, int geometry_counters);

/* Borrowed DEVICE pointers, valid until the next loc_simulate:
 *   counters: float [ncell][ntrans_padded][2]; slot k of a cell belongs to the k-th selected transition:
 *       [k][0] = SJ  = sum over ray steps of (a s / V_eff) sum_c phi_c n_c (1-e^-tau_c)/tau_c, n_c the photon
 *                occupation number I_c c^2 / (2 h nu^3) entering the step: the profile- and path-weighted mean
 *                radiation field.  Absorbed-photon count of Eq. 2:  ABS = k_t V_eff (4 pi dv / h c)(2 h nu^3/c^2) SJ.
 *       [k][1] = ESC = sum over steps of (a s / V_eff) [ (1 - sum_c phi_c) + sum_c phi_c (1-e^-tau_c)/tau_c ]
 *                = escape probability of the cell's own photons = 1 - LAMBDA* (PAPER.md:81).
 *   visits:   uint32 [ncell] ray segments per cell        (only if geometry_counters)
 *   pathz:    uint32 [ncell] summed main-axis path in grid units, 2^20 per root cell (octree, geometry_counters)
 * Photon counts themselves (~1e38 per second for parsec-size cells) do not fit float32; see DESIGN.md 5.2. */
int loc_get_counters(loc_model *m, const float **counters, int *ntrans_padded, const uint32_t **visits,
                     const uint32_t **pathz);

/* Per-cell statistical equilibrium; LOC_ESTATE before the first loc_simulate (the counters hold nothing),
 * LOC_ENONFINITE if a population came out NaN / infinite.  S_lu = (g_u/g_l) A SJ replaces B_lu I, A_ul is scaled by
 * ESC, collisions from `density` and `tkin`; transitions that were not traced see the background only
 * (DESIGN R23).  Writes the new populations into the registered buffer and refreshes the line coefficients.
 * max_rel_change (host, may be NULL): largest relative change over levels holding >= 1e-10 of the molecules. */
int loc_solve(loc_model *m, double *max_rel_change);

/* niter x (loc_simulate with the remembered selection; loc_solve); no early exit.  niter = 0 runs nothing
 * and reports a change of 0.                                                                              */
int loc_iterate(loc_model *m, int niter, double *max_rel_change);

/* ali = 1 (default): accelerated lambda iteration -- loc_solve scales A_ul by the escape probability ESC and uses the
 * radiation field of the other cells only.  ali = 0: plain lambda iteration ("it is also possible to run
 * LOC without ALI"): A_ul unscaled, and the self term of Eq. 2 is kept, i.e. the photons a
 * cell absorbs from its own emission, (1 - ESC) times the source function of the populations the rays were traced
 * with, are added to SJ.  Both modes share loc_simulate and its counters and have the same fixed point; only
 * loc_solve differs.  Returns LOC_EINVAL for any other value.                                                */
int loc_set_ali(loc_model *m, int ali);

/* Accuracy / launch knobs (keys LOC_OPT_* above).  LOC_EINVAL for an unknown key or a value outside the key's range.
 * Channel widths: loc_simulate and loc_spectra need no minimum resolution of the line profile -- with channels wider than
 * the line (dv > sigma) the sampled profile of PAPER.md:73 is no longer normalised, and the kernels then sum the sampled
 * values themselves instead of using the analytic wing mass, and widen the window by 2 ln (dv/sigma)^2.
 * ITERATION is another matter: for dv > 2 sigma the sampled profile can sum to more than 1, the method's own LAMBDA*
 * then exceeds 1 (ESC < 0) and the accelerated rate equations leave the physical range -- in the float64
 * oracle just as in the kernels.  loc_solve / loc_iterate* are defined for dv <= 2 sigma in every cell; beyond that their
 * result is unspecified (it may be LOC_ENONFINITE).  The counters of a single loc_simulate stay well defined.          */
int loc_set_option(loc_model *m, int key, double value);

/* Convergence-controlled iteration ("repeated until the level populations converge"):
 * (loc_simulate; loc_solve) until max_rel_change <= tol or max_iter iterations were done.  niter_done (host, may be
 * NULL) receives the number of iterations run, max_rel_change (host, may be NULL) the change of the last one.
 * Synchronises the stream once per iteration.  max_iter = 0 runs nothing and reports a change of 0.          */
int loc_iterate_until(loc_model *m, int max_iter, double tol, int *niter_done, double *max_rel_change);

/* Spectral map: for each pixel one line of sight through the model with the current
 * populations, T_A(c) = (c^2 / 2 k nu^2)(I_c - B_nu(T_bg)), written to dev_out float [ny][nx][nchannel] (K).
 * Octree: lines of sight run along `dir` (host double[3]); pixel (ix,iy) starts on the upstream face at the
 * integer grid position  (aff[0] + ix aff[2] + iy aff[3],  aff[1] + ix aff[4] + iy aff[5])  of the two transverse
 * axes (units: 2^20 per root cell, in the ray's working frame, DESIGN 6.4).
 * Shells: dir = NULL, ny = 1, pixel ix is the line of sight with impact parameter offsets_cm[ix] (host).   */
int loc_spectra(loc_model *m, int trans, const double *dir, int nx, int ny, const int64_t *aff,
                const double *offsets_cm, float *dev_out);

/* The same map in the CALLER's frame (octree models; "pixel = smallest cell"): model coordinates in cm with
 * the origin at the corner of root cell (0,0,0).  `dir` (host double[3], unit) is the direction the photons travel, i.e.
 * from the far side of the model towards the observer.  The image plane is spanned by e2 = the unit projection of "north"
 * perpendicular to dir (north = +z; +y when dir is parallel to z within 1e-9) and e1 = e2 x dir; pixel (ix, iy), ix fastest,
 * is the line of sight through
 *     X(ix, iy) = centre_cm + (ix - (nx-1)/2) pixel_cm e1 + (iy - (ny-1)/2) pixel_cm e2 .
 * (dir = +z: e1 = +x, e2 = +y.)  The library snaps dir to its fixed-point slopes (DESIGN R7) and converts X to the integer
 * start position on the upstream face; lines of sight that miss the model return the zero spectrum.
 * dev_out: DEVICE float [ny][nx][nchannel] (K).                                                                         */
int loc_spectra_map(loc_model *m, int trans, const double *dir, int nx, int ny, double pixel_cm, const double *centre_cm,
                    float *dev_out);

/* Excitation temperature of transition `trans` in every cell from the current populations (Fig. 4: the
 * quantity whose change per iteration and per density bin the paper uses to judge convergence; the binning is left to
 * the caller):  T_ex = -(h nu / k) / ln(n_u g_l / (n_l g_u)), K.  dev_tex: DEVICE float [ncell]; 0 in refined (non-leaf)
 * cells and in cells without molecules.  Enqueued on the model's stream.                                        */
int loc_tex(loc_model *m, int trans, float *dev_tex);

/* Line-area map (Fig. 5c "line area"): W[p] = sum_c T_A[p][c] * dv, in K km/s, for npix spectra of the
 * model's nchannel channels as loc_spectra writes them.  dev_cube: DEVICE float [npix][nchannel] (K); dev_w: DEVICE
 * float [npix].  Enqueued on the model's stream; npix = 0 is a no-op.                                          */
int loc_line_area(loc_model *m, const float *dev_cube, int64_t npix, float *dev_w);

/* Spectra of a shell model for callers that cannot allocate device memory.
 *
 * Everything else in this header needs a loc_model, and a loc_model needs a workspace that somebody obtained from
 * cudaMalloc (or a pool built on it).  Some code that wants a spectrum is not in a position to do that: a plug-in or
 * callback that is handed its input and output buffers by a host application which owns every byte of device memory; a
 * monitoring or display step that runs next to a solver whose workspace already fills the GPU; code on a latency-critical
 * path where the implicit device-wide synchronisation of cudaMalloc / cudaFree is not acceptable.  For those callers this
 * one call computes what loc_spectra computes for a LOC_GRID_SHELL model (PAPER.md:77 line-of-sight integration,
 * PAPER.md:137 Doppler shift from the direction cosine at the entry of each step; same kernel, k_spectra1d) from plain
 * arrays, without a model and without a workspace.  The scratch the kernel needs -- a device copy of the shell radii and
 * the packed (radial velocity, total line width) record per shell -- lives in a fixed array inside the library image of
 * 24 * LOC_STATIC_MAX_SHELLS bytes (96 KiB), which every GPU that loads the library holds until the process exits.
 * The call itself allocates nothing: no cudaMalloc / cudaFree, no allocating library routine.
 *
 *   nshell            1 .. LOC_STATIC_MAX_SHELLS; more shells -> LOC_EINVAL with a message that names the limit (use a
 *                     loc_model with a workspace for larger models)
 *   r_out             host [nshell], strictly ascending, cm (as in loc_grid); copied during the call
 *   dev_vrad, dev_sigma, dev_tkin
 *                     DEVICE float [nshell]: radial velocity (cm/s, positive outward), turbulent 1-D velocity dispersion
 *                     (cm/s) and kinetic temperature (K), as in loc_cells; the thermal width k T / m is added for
 *                     mass_amu > 0 (mass_amu = 0: dev_sigma is the total width, DESIGN R3)
 *   dev_pop_u, dev_pop_l
 *                     DEVICE float [nshell]: populations (cm^-3) of the upper and lower level of the line
 *   freq_hz, einstein_A, g_upper, g_lower
 *                     the line: rest frequency (Hz), Einstein A (1/s), statistical weights.  No hyperfine structure.
 *   nchannel, band_halfwidth_cm_s, t_background_K
 *                     as in loc_create_model (1 <= nchannel <= 1024)
 *   nlos, offsets_cm  host [nlos]: impact parameters of the lines of sight (cm; the sign is ignored; beyond the outer
 *                     radius the spectrum is zero).  nlos = 0 is a no-op.
 *   dev_out           DEVICE float [nlos][nchannel]: T_A in K, as loc_spectra writes it
 *   stream            cudaStream_t as void* (NULL = default stream) of the CURRENT device; all work is enqueued there and
 *                     the call does not wait for it
 *   err, err_len      optional host buffer that receives the text of a failure (may be NULL)
 *
 * Rules that follow from the shared array:
 *   - The first call on a device looks up the array's address on that device (cudaGetSymbolAddress, with that device
 *     current) and remembers it.  Make that first call during start-up, before any stream capture is begun.
 *   - All calls on a device use the same array.  Calls on one stream are ordered and safe back to back.  Calls whose GPU
 *     work can overlap (different streams without an event between them, or several host threads each with a stream of
 *     its own) race on the array and give wrong spectra: serialise them.
 *   - The array keeps what the last call wrote.  Each call overwrites the entries it reads (the first nshell) before
 *     reading them, so nothing needs clearing and a smaller model after a larger one is safe.
 * Returns LOC_OK, LOC_EINVAL (bad argument or size) or LOC_ECUDA.                                                       */
#define LOC_STATIC_MAX_SHELLS 4096
int loc_spectra_shells_static(int nshell, const double *r_out, const float *dev_vrad, const float *dev_sigma,
                              const float *dev_tkin, double mass_amu, const float *dev_pop_u, const float *dev_pop_l,
                              double freq_hz, double einstein_A, double g_upper, double g_lower, int nchannel,
                              double band_halfwidth_cm_s, double t_background_K, int nlos, const double *offsets_cm,
                              float *dev_out, void *stream, char *err, int err_len);

int loc_get_stats(loc_model *m, loc_stats *out);
void loc_destroy_model(loc_model *m);
const char *loc_last_error(const loc_model *m); /* m may be NULL: error of the last failed loc_create_model */

#ifdef __cplusplus
}
#endif
#endif /* LOC_H */
