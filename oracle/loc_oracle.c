/*
 * loc_oracle.c -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * A plain, slow, double-precision CPU restatement of the line radiative
 * transfer step of LOC (arxiv 2009.12609, M. Juvela), written from the paper's
 * equations so that the CUDA library can be checked against it.  It shares no
 * code with paper_2009_12609_b200/csrc and is never imported by the product.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * Citations are PAPER.md:<line> and the readings
 * R1..Rn listed in DESIGN.md section 3 ("Readings of the paper").
 *
 * Every channel is evaluated (no profile cut-off), every sum is a plain loop.
 * The optional OpenMP pragmas only distribute whole rays over threads and add
 * to the counters with atomic double adds (3D) or into per-thread counters that
 * are summed in thread order (1D, round 3); the arithmetic per ray is serial.
 *
 * Pins (tests/test_oracle_*.py): slab closed form, optically thin limit, LTE
 * limit, blackbody enclosure, two-level closed form, photon ledger, path
 * invariants, ALI == Lambda fixed point, brute-force ray/box geometry, full
 * refinement == finer grid, mirror symmetry, GTH cross-check of the solver;
 * since round 2 also: collision-rate interpolation against numpy.interp
 * (nodes, midpoints, clamps), the untraced-transition branch of orc_solve
 * (two-level closed form with nsel = 0; thin limit), the entry cosine of the
 * 1D path (mu r_entry = ray abscissa), the donor spectrum at ray births on a
 * layered model with partial refinement (every level's leaves == the uniform
 * Cartesian grid of that resolution), the thick closed form of orc_spectra_1d,
 * 90-degree rotation / z-mirror of the direction set in 3D; since round 3 the
 * side entry and side exit of a map's lines of sight (orc_spectra_3d: path
 * inside the uniform model from the lattice definition by integer search).
 * Hyperfine structure (profile_t): tests/test_oracle_pins_hfs.py; sub-iterations (orc_solve_sub): tests/test_oracle_subiter.py.
 * Parity unpinned: none of the functions below.  One READING stays constrained
 * by invariants only (blackbody enclosure P4, ledger P6): at a SIDE-face birth
 * the donor is the line that entered the level-(tag-1) ancestor through its
 * upstream face (R9/R10) -- the paper's text fixes no
 * more than that, and no closed form distinguishes the transverse choice.
 * (Absolute T_ex profiles of the paper's figures are not reproducible: their
 * inputs are not available.)
 */
#ifdef _OPENMP
#include <omp.h>
#endif
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---- O1 constants (CGS, CODATA 2018); the paper gives none (reading R1) ---- */
#define ORC_H 6.62607015e-27
#define ORC_K 1.380649e-16
#define ORC_C 2.99792458e10
#define ORC_AMU 1.66053906660e-24
#define ORC_PI 3.14159265358979323846

typedef struct {
    int nlevel;
    const double *energy_K; /* [nlevel] E_i / k                         */
    const double *g;        /* [nlevel] statistical weights             */
    int ntrans;
    const int *upper; /* [ntrans]                                      */
    const int *lower; /* [ntrans]                                      */
    const double *A;  /* [ntrans] Einstein A (1/s)                      */
    double mass_amu;  /* 0 -> sigma input is the total width (R3)       */
    int ncoll;
    const int *cu; /* [ncoll] upper level of collisional pair        */
    const int *cl; /* [ncoll] lower level                            */
    int ntemp;
    const double *temps_K;   /* [ntemp] ascending                        */
    const double *rate_down; /* [ntemp][ncoll] cm^3/s                    */
    /* hyperfine structure with LTE between the components: transition t has the
     * components hf_off[t] .. hf_off[t+1]-1, each a Gaussian of the cell's width shifted by hf_dv (cm/s, on the channel
     * velocity axis) carrying the fraction hf_w of the line (sum = 1).  One population per level: the components share
     * the source function.  hf_off == NULL or an empty range: a single component at zero offset.                      */
    const int *hf_off;    /* [ntrans+1] or NULL */
    const double *hf_dv;  /* [hf_off[ntrans]] */
    const double *hf_w;   /* [hf_off[ntrans]] */
} orc_species;

/* ledger slots (pin P6) */
enum { LG_INJECTED = 0, LG_EMITTED, LG_CREATED, LG_ABSORBED, LG_SELFABS, LG_ESCAPED, LG_TERMINATED, LG_RESCALE, LG_N };

/* Planck function B_nu(T), erg s^-1 cm^-2 Hz^-1 sr^-1 */
double orc_planck(double nu, double T)
{
    if (T <= 0.0) return 0.0;
    return 2.0 * ORC_H * nu * nu * nu / (ORC_C * ORC_C) / expm1(ORC_H * nu / (ORC_K * T));
}

/* line frequency from level energies (O2) */
double orc_freq(const orc_species *sp, int t)
{
    return (sp->energy_K[sp->upper[t]] - sp->energy_K[sp->lower[t]]) * ORC_K / ORC_H;
}

/* O3: LTE populations at T_kin ("calculations start with LTE conditions") */
void orc_lte(const orc_species *sp, int64_t ncell, const double *density, const double *tkin,
             const double *abundance, double *pops /* [ncell][nlevel] */)
{
    int NL = sp->nlevel;
    for (int64_t c = 0; c < ncell; c++) {
        double Z = 0.0;
        for (int i = 0; i < NL; i++) Z += sp->g[i] * exp(-sp->energy_K[i] / tkin[c]);
        for (int i = 0; i < NL; i++)
            pops[c * NL + i] = density[c] * abundance[c] * sp->g[i] * exp(-sp->energy_K[i] / tkin[c]) / Z;
    }
}

/* O2: downward rate coefficient of pair k at temperature T: linear interpolation, clamped (R18) */
static double coll_gamma(const orc_species *sp, int k, double T)
{
    int nt = sp->ntemp;
    if (nt == 1 || T <= sp->temps_K[0]) return sp->rate_down[k];
    if (T >= sp->temps_K[nt - 1]) return sp->rate_down[(size_t)(nt - 1) * sp->ncoll + k];
    int j = 0;
    while (T > sp->temps_K[j + 1]) j++;
    double f = (T - sp->temps_K[j]) / (sp->temps_K[j + 1] - sp->temps_K[j]);
    return (1.0 - f) * sp->rate_down[(size_t)j * sp->ncoll + k] + f * sp->rate_down[(size_t)(j + 1) * sp->ncoll + k];
}

/* Rate matrix R[i*NL+j] = rate i->j (1/s) for one cell (O9).
 *   S_t  = induced upward rate ("S_lu is used directly in place of B_lu I")
 *   beta = escape probability scaling A_ul                               */
static void build_rates(const orc_species *sp, double n, double T, const double *S, const double *beta, double *R)
{
    int NL = sp->nlevel;
    memset(R, 0, sizeof(double) * NL * NL);
    for (int t = 0; t < sp->ntrans; t++) {
        int u = sp->upper[t], l = sp->lower[t];
        R[u * NL + l] += sp->A[t] * beta[t] + S[t] * sp->g[l] / sp->g[u];
        R[l * NL + u] += S[t];
    }
    for (int k = 0; k < sp->ncoll; k++) {
        int u = sp->cu[k], l = sp->cl[k];
        double gd = coll_gamma(sp, k, T);
        double gu = gd * sp->g[u] / sp->g[l] * exp(-(sp->energy_K[u] - sp->energy_K[l]) / T);
        R[u * NL + l] += n * gd;
        R[l * NL + u] += n * gu;
    }
}

/* O9: Gaussian elimination with partial pivoting of  M x = b, M_ij = R[j->i], M_ii = -sum_j R[i->j],
 * last row replaced by ones, b = (0,...,0,ntot).  Returns 0 on success.                            */
static int solve_ge(int NL, const double *R, double ntot, double *x)
{
    double M[32 * 33];
    if (NL > 32) return -1;
    int W = NL + 1;
    for (int i = 0; i < NL; i++) {
        for (int j = 0; j < NL; j++) M[i * W + j] = (i == j) ? 0.0 : R[j * NL + i];
        double s = 0.0;
        for (int j = 0; j < NL; j++)
            if (j != i) s += R[i * NL + j];
        M[i * W + i] = -s;
        M[i * W + NL] = 0.0;
    }
    for (int j = 0; j < NL; j++) M[(NL - 1) * W + j] = 1.0;
    M[(NL - 1) * W + NL] = ntot;
    for (int c = 0; c < NL; c++) {
        int piv = c;
        for (int r = c + 1; r < NL; r++)
            if (fabs(M[r * W + c]) > fabs(M[piv * W + c])) piv = r;
        if (M[piv * W + c] == 0.0) return -2;
        if (piv != c)
            for (int j = 0; j <= NL; j++) {
                double tmp = M[c * W + j];
                M[c * W + j] = M[piv * W + j];
                M[piv * W + j] = tmp;
            }
        for (int r = c + 1; r < NL; r++) {
            double f = M[r * W + c] / M[c * W + c];
            for (int j = c; j <= NL; j++) M[r * W + j] -= f * M[c * W + j];
        }
    }
    for (int i = NL - 1; i >= 0; i--) {
        double s = M[i * W + NL];
        for (int j = i + 1; j < NL; j++) s -= M[i * W + j] * x[j];
        x[i] = s / M[i * W + i];
    }
    return 0;
}

/* Independent second algorithm used only as a pin of solve_ge (tests): Grassmann-Taksar-Heyman
 * subtraction-free stationary distribution of the same rate matrix.                              */
int orc_solve_gth(int NL, const double *Rin, double ntot, double *x)
{
    double R[32 * 32];
    if (NL > 32) return -1;
    memcpy(R, Rin, sizeof(double) * NL * NL);
    for (int n = NL - 1; n >= 1; n--) {
        double s = 0.0;
        for (int j = 0; j < n; j++) s += R[n * NL + j];
        if (s <= 0.0) return -2;
        for (int i = 0; i < n; i++) R[i * NL + n] /= s;
        for (int i = 0; i < n; i++)
            for (int j = 0; j < n; j++)
                if (i != j) R[i * NL + j] += R[i * NL + n] * R[n * NL + j];
    }
    x[0] = 1.0;
    double tot = 1.0;
    for (int n = 1; n < NL; n++) {
        double s = 0.0;
        for (int i = 0; i < n; i++) s += x[i] * R[i * NL + n];
        x[n] = s;
        tot += s;
    }
    for (int i = 0; i < NL; i++) x[i] *= ntot / tot;
    return 0;
}

/* expose the rate matrix and the GE solve for the pins */
void orc_rate_matrix(const orc_species *sp, double n, double T, const double *S, const double *beta, double *R)
{
    build_rates(sp, n, T, S, beta, R);
}
int orc_solve_rates(int NL, const double *R, double ntot, double *x) { return solve_ge(NL, R, ntot, x); }

/* O9 over all cells.
 *   P   [nsel][ncell]  path-form absorbed-photon counter  (Eq. 2 first term / k_t)
 *   LAM [nsel][ncell]  fraction of the cell's own photons re-absorbed in the cell
 *   veff[ncell]        sampled cell volume (reading R12)
 *   sel [nsel]         which transitions were ray traced; the others use background only (R23)
 * returns max relative population change over levels with n_i/sum >= 1e-10 (R20).               */
double orc_solve(const orc_species *sp, int64_t ncell, const double *density, const double *tkin,
                 const double *abundance, const double *veff, int nsel, const int *sel, const double *P,
                 const double *LAM, double dv, double tbg, int ali, double *pops /* in/out [ncell][NL] */)
{
    int NL = sp->nlevel, NT = sp->ntrans;
    double maxrel = 0.0;
    int *slot = (int *)malloc(sizeof(int) * NT);
    for (int t = 0; t < NT; t++) slot[t] = -1;
    for (int k = 0; k < nsel; k++) slot[sel[k]] = k;
#pragma omp parallel for reduction(max : maxrel) schedule(static)
    for (int64_t c = 0; c < ncell; c++) {
        double S[64], beta[64], R[32 * 32], x[32];
        double ntot = density[c] * abundance[c];
        if (ntot <= 0.0) {
            for (int i = 0; i < NL; i++) pops[c * NL + i] = 0.0;
            continue;
        }
        for (int t = 0; t < NT; t++) {
            int u = sp->upper[t], l = sp->lower[t];
            double nu = orc_freq(sp, t);
            double gr = sp->g[u] / sp->g[l];
            if (slot[t] >= 0) {
                /* S_lu = (g_u/g_l) c^3 A /(8 pi nu^3 dv) * P / V   (O9; equals B_lu * Jbar) */
                double coef = gr * ORC_C * ORC_C * ORC_C * sp->A[t] / (8.0 * ORC_PI * nu * nu * nu * dv);
                S[t] = coef * P[(size_t)slot[t] * ncell + c] / veff[c];
                beta[t] = ali ? 1.0 - LAM[(size_t)slot[t] * ncell + c] : 1.0;
            } else {
                /* R23: not ray traced -> optically thin, background radiation only */
                S[t] = (tbg > 0.0) ? gr * sp->A[t] / expm1(ORC_H * nu / (ORC_K * tbg)) : 0.0;
                beta[t] = 1.0;
            }
        }
        build_rates(sp, density[c], tkin[c], S, beta, R);
        solve_ge(NL, R, ntot, x);
        for (int i = 0; i < NL; i++) {
            double old = pops[c * NL + i];
            if (x[i] / ntot >= 1e-10 || old / ntot >= 1e-10) {
                double rel = fabs(x[i] - old) / fmax(fabs(x[i]), 1e-300);
                if (rel > maxrel) maxrel = rel;
            }
            pops[c * NL + i] = x[i];
        }
    }
    free(slot);
    return maxrel;
}

/* Sub-iterations of the solve between two ray passes ("some form of sub-iterations, where level
 * populations are updated more frequently in optically thick regions" -- the paper gives no formula: DESIGN.md R26).
 * The ray pass measured, per cell and traced transition, the escape probability beta0 = 1 - LAM and the external field P with
 * the OLD populations.  A one-zone model of the cell carries both to other populations: tau_eff is defined by
 * E(tau_eff) = beta0, E(tau) = (1 - e^-tau)/tau; new populations change the line opacity by r = k_new / k_old
 * (k = n_l g_u/g_l - n_u), and then beta = E(tau_eff r), P = P0 beta / beta0 (the external photons meet the same escape
 * probability on their way in).  Sub-iteration 1 is the plain ALI solve (r = 1); each further one re-solves with (beta, P) of
 * the previous solution.  At the ALI fixed point r = 1, so the fixed point is unchanged.  nsub = 1 == orc_solve.         */
static double e_of_tau(double t) { return (fabs(t) < 1e-6) ? 1.0 - t / 2.0 + t * t / 6.0 : -expm1(-t) / t; }
static double inv_e(double beta) /* tau >= 0 with E(tau) = beta, by bisection (E is decreasing) */
{
    if (!(beta < 1.0)) return 0.0;
    if (!(beta > 0.0)) return 1e300;
    double lo = 0.0, hi = 2.0 / beta + 1.0;
    for (int i = 0; i < 200; i++) {
        double mid = 0.5 * (lo + hi);
        if (e_of_tau(mid) > beta) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}
double orc_solve_sub(const orc_species *sp, int64_t ncell, const double *density, const double *tkin,
                     const double *abundance, const double *veff, int nsel, const int *sel, const double *P,
                     const double *LAM, double dv, double tbg, int nsub, double *pops /* in/out [ncell][NL] */)
{
    int NL = sp->nlevel, NT = sp->ntrans;
    double maxrel = 0.0;
    int *slot = (int *)malloc(sizeof(int) * NT);
    for (int t = 0; t < NT; t++) slot[t] = -1;
    for (int k = 0; k < nsel; k++) slot[sel[k]] = k;
#pragma omp parallel for reduction(max : maxrel) schedule(static)
    for (int64_t c = 0; c < ncell; c++) {
        double S0[64], S[64], beta0[64], beta[64], teff[64], k0[64], R[32 * 32], x[32];
        double ntot = density[c] * abundance[c];
        if (ntot <= 0.0) {
            for (int i = 0; i < NL; i++) pops[c * NL + i] = 0.0;
            continue;
        }
        for (int t = 0; t < NT; t++) {
            int u = sp->upper[t], l = sp->lower[t];
            double nu = orc_freq(sp, t);
            double gr = sp->g[u] / sp->g[l];
            k0[t] = pops[c * NL + l] * gr - pops[c * NL + u];
            if (slot[t] >= 0) {
                double coef = gr * ORC_C * ORC_C * ORC_C * sp->A[t] / (8.0 * ORC_PI * nu * nu * nu * dv);
                S0[t] = coef * P[(size_t)slot[t] * ncell + c] / veff[c];
                beta0[t] = 1.0 - LAM[(size_t)slot[t] * ncell + c];
                teff[t] = inv_e(beta0[t]);
            } else {
                S0[t] = (tbg > 0.0) ? gr * sp->A[t] / expm1(ORC_H * nu / (ORC_K * tbg)) : 0.0;
                beta0[t] = 1.0;
                teff[t] = 0.0;
            }
            S[t] = S0[t];
            beta[t] = beta0[t];
        }
        for (int it = 0; it < nsub; it++) {
            build_rates(sp, density[c], tkin[c], S, beta, R);
            solve_ge(NL, R, ntot, x);
            for (int t = 0; t < NT; t++) {
                if (slot[t] < 0 || !(beta0[t] > 0.0) || k0[t] == 0.0) continue;
                int u = sp->upper[t], l = sp->lower[t];
                double r = (x[l] * sp->g[u] / sp->g[l] - x[u]) / k0[t];
                if (!(r > 0.0)) r = 1.0; /* inverted or vanishing line: keep the measured values */
                beta[t] = e_of_tau(teff[t] * r);
                S[t] = S0[t] * beta[t] / beta0[t];
            }
        }
        for (int i = 0; i < NL; i++) {
            double old = pops[c * NL + i];
            if (x[i] / ntot >= 1e-10 || old / ntot >= 1e-10) {
                double rel = fabs(x[i] - old) / fmax(fabs(x[i]), 1e-300);
                if (rel > maxrel) maxrel = rel;
            }
            pops[c * NL + i] = x[i];
        }
    }
    free(slot);
    return maxrel;
}

/* T_ex of transition t from populations (O9) */
double orc_tex(const orc_species *sp, int t, double nu_pop, double nl_pop)
{
    int u = sp->upper[t], l = sp->lower[t];
    double r = nu_pop * sp->g[l] / (nl_pop * sp->g[u]);
    return -(ORC_H * orc_freq(sp, t) / ORC_K) / log(r);
}

/* ------------------------------------------------------------------------------------------
 * O4 profile and O6 cell step
 * ---------------------------------------------------------------------------------------- */

/* phi_c = dv/(sigma sqrt(2 pi)) exp(-(v_c - v0)^2 / (2 sigma^2)): "fraction of emitted photons per
 * channel", not renormalised, not truncated (R13).  v_c = (c-(NCH-1)/2) dv.            */
static void profile(int nch, double dv, double sigma, double v0, double *phi)
{
    double amp = dv / (sigma * sqrt(2.0 * ORC_PI));
    for (int c = 0; c < nch; c++) {
        double vc = (c - 0.5 * (nch - 1)) * dv;
        double x = (vc - v0) / sigma;
        phi[c] = amp * exp(-0.5 * x * x);
    }
}

/* Profile of transition t: the sum over its hyperfine components  phi_c = sum_k w_k dv/(sigma sqrt(2 pi)) exp(-(v_c - v0 -
 * dv_k)^2 / (2 sigma^2))  (LTE between the components: PAPER.md:39, 149); without hyperfine structure the plain profile. */
static void profile_t(const orc_species *sp, int t, int nch, double dv, double sigma, double v0, double *phi)
{
    if (!sp->hf_off || sp->hf_off[t + 1] == sp->hf_off[t]) {
        profile(nch, dv, sigma, v0, phi);
        return;
    }
    double amp = dv / (sigma * sqrt(2.0 * ORC_PI));
    for (int c = 0; c < nch; c++) phi[c] = 0.0;
    for (int k = sp->hf_off[t]; k < sp->hf_off[t + 1]; k++)
        for (int c = 0; c < nch; c++) {
            double vc = (c - 0.5 * (nch - 1)) * dv;
            double x = (vc - v0 - sp->hf_dv[k]) / sigma;
            phi[c] += sp->hf_w[k] * amp * exp(-0.5 * x * x);
        }
}

static double total_sigma(const orc_species *sp, double sigma_turb, double T)
{
    if (sp->mass_amu <= 0.0) return sigma_turb;
    return sqrt(sigma_turb * sigma_turb + ORC_K * T / (sp->mass_amu * ORC_AMU)); /* R3 */
}

/* f = (1-e^-tau)/tau and 1-f, with series for tiny |tau| (O6) */
static void f_of_tau(double tau, double *f, double *omf)
{
    if (fabs(tau) < 1e-5) {
        *f = 1.0 - tau / 2.0 + tau * tau / 6.0 - tau * tau * tau / 24.0;
        *omf = tau / 2.0 - tau * tau / 6.0 + tau * tau * tau / 24.0;
    } else {
        *f = -expm1(-tau) / tau;
        *omf = 1.0 - *f;
    }
}

/* One cell step of one ray for one transition (O6).
 *   N[nch]  photons per second per channel carried by the ray, updated by Eq. 3
 *   a       ray weight (cm^2), s step length (cm), veff sampled cell volume (cm^3)
 *   accumulates ABS (Eq. 2 first term, net absorbed external photons), P (path form), LAM
 *   ali == 0: the self term of Eq. 2 with the 1/tau of reading R2 is added to P as well.            */
static void cell_step(int nch, double *N, const double *phi, double a, double s, double veff, double kcoef /* c^3 A/(8 pi nu^3 dv) */,
                      double gr /* g_u/g_l */, double A, double n_u, double n_l, int ali, double *ABS, double *P,
                      double *LAM, double *ledger)
{
    double kt = kcoef * (n_l * gr - n_u); /* cm^-1 per unit phi */
    double abs_sum = 0.0, p_sum = 0.0, lam_sum = 0.0;
    double em_sum = 0.0, self_sum = 0.0;
    for (int c = 0; c < nch; c++) {
        double tau = kt * phi[c] * s;
        double f, omf;
        f_of_tau(tau, &f, &omf);
        double ome = tau * f; /* 1 - e^-tau without cancellation */
        double emit = n_u * A * (a * s) * phi[c]; /* this ray's share a*s/V of n_u A V phi */
        abs_sum += N[c] * ome;
        p_sum += s * phi[c] * N[c] * f;
        lam_sum += (a * s / veff) * phi[c] * omf;
        if (!ali) {
            /* R2: self term  n_u A V phi (1/tau)[1 - (1-e^-tau)/tau]  in path form */
            double g2 = (fabs(tau) < 1e-5) ? 0.5 - tau / 6.0 + tau * tau / 24.0 : omf / tau;
            p_sum += s * phi[c] * emit * g2;
        }
        em_sum += emit;
        self_sum += emit * omf;
        N[c] = N[c] * (1.0 - ome) + emit * f; /* Eq. 3 */
    }
#pragma omp atomic
    *ABS += abs_sum;
#pragma omp atomic
    *P += p_sum;
#pragma omp atomic
    *LAM += lam_sum;
    if (ledger) {
        ledger[LG_ABSORBED] += abs_sum;
        ledger[LG_EMITTED] += em_sum;
        ledger[LG_SELFABS] += self_sum;
    }
}

/* Eq. 1 with A cos(theta) Omega -> a * 4 pi (O5): background photons per channel */
static double bg_photons(double nu, double tbg, double a, double dv)
{
    return orc_planck(nu, tbg) * a * 4.0 * ORC_PI * dv / (ORC_H * ORC_C);
}

/* ------------------------------------------------------------------------------------------
 * O7: one-dimensional (spherically symmetric) models
 * ---------------------------------------------------------------------------------------- */

/* shell index containing impact parameter p: r_{k-1} <= p < r_k */
static int shell_of(int ns, const double *r, double p)
{
    int k = 0;
    while (k < ns - 1 && p >= r[k]) k++;
    return k;
}

/* path table of one ray: fills seg_shell[], seg_s[], seg_mu[]; returns number of segments (O7, R5) */
static int ray_path_1d(int ns, const double *r, double p, int *seg_shell, double *seg_s, double *seg_mu)
{
    int k0 = shell_of(ns, r, p);
    int n = 0;
    for (int k = ns - 1; k > k0; k--) { /* inbound */
        seg_shell[n] = k;
        seg_s[n] = sqrt(r[k] * r[k] - p * p) - sqrt(r[k - 1] * r[k - 1] - p * p);
        seg_mu[n] = -sqrt(1.0 - p * p / (r[k] * r[k]));
        n++;
    }
    seg_shell[n] = k0; /* tangent shell: one step (R5) */
    seg_s[n] = 2.0 * sqrt(r[k0] * r[k0] - p * p);
    seg_mu[n] = -sqrt(1.0 - p * p / (r[k0] * r[k0]));
    n++;
    for (int k = k0 + 1; k < ns; k++) { /* outbound */
        seg_shell[n] = k;
        seg_s[n] = sqrt(r[k] * r[k] - p * p) - sqrt(r[k - 1] * r[k - 1] - p * p);
        seg_mu[n] = sqrt(1.0 - p * p / (r[k - 1] * r[k - 1]));
        n++;
    }
    return n;
}

/* sampled shell volumes V_eff,k = sum_i W_i s_ik (R12); also returns per-ray segment counts */
void orc_veff_1d(int ns, const double *r, int nray, const double *p, const double *w, double *veff)
{
    int *sh = (int *)malloc(sizeof(int) * 2 * ns);
    double *ss = (double *)malloc(sizeof(double) * 2 * ns), *mu = (double *)malloc(sizeof(double) * 2 * ns);
    for (int k = 0; k < ns; k++) veff[k] = 0.0;
    for (int i = 0; i < nray; i++) {
        int n = ray_path_1d(ns, r, p[i], sh, ss, mu);
        for (int j = 0; j < n; j++) veff[sh[j]] += w[i] * ss[j];
    }
    free(sh);
    free(ss);
    free(mu);
}

/* copy of the path table for the pins (P7) */
int orc_path_1d(int ns, const double *r, double p, int *seg_shell, double *seg_s, double *seg_mu)
{
    return ray_path_1d(ns, r, p, seg_shell, seg_s, seg_mu);
}

/* O5-O7 simulation of all rays for the selected transitions.
 * Outputs [nsel][ns]: ABS, P, LAM; visits[ns]; ledger[LG_N]; optionally the emerging photon
 * vectors nout[nray][nsel][nch] (used by the slab / thin pins).                                       */
int orc_sim_1d(const orc_species *sp, int ns, const double *r, const double *tkin, const double *sigma_turb,
               const double *vrad, int nray, const double *p, const double *w, const double *pops /*[ns][NL]*/,
               int nch, double band_half, double tbg, int nsel, const int *sel, int ali, double *ABS, double *P,
               double *LAM, int64_t *visits, double *ledger, double *nout)
{
    int NL = sp->nlevel;
    double dv = 2.0 * band_half / nch;
    double *veff = (double *)malloc(sizeof(double) * ns);
    orc_veff_1d(ns, r, nray, p, w, veff);
    memset(ABS, 0, sizeof(double) * nsel * ns);
    memset(P, 0, sizeof(double) * nsel * ns);
    memset(LAM, 0, sizeof(double) * nsel * ns);
    if (visits) memset(visits, 0, sizeof(int64_t) * ns);
    if (ledger) memset(ledger, 0, sizeof(double) * LG_N);
    /* Whole rays are dealt out to the threads in turn (schedule(static, 1): ray i goes to thread i mod T -- the rays
     * differ in length by the number of shells they cross, and dealing balances that); every thread adds into counters of
     * its own, and the threads' counters are added up in thread order afterwards.  The arithmetic per ray is serial and in
     * the paper's order; with one thread the sums are those of the plain loop over rays, bit for bit; with T threads only
     * the order in which the rays' contributions to a shell are added differs (rounding, ~1e-16 relative).             */
    int nthr = 1;
#ifdef _OPENMP
    nthr = omp_get_max_threads();
    if (nthr > nray) nthr = nray;
    if (nthr < 1) nthr = 1;
#endif
    size_t ncnt = (size_t)nsel * ns;
    double *tacc = (double *)calloc((size_t)nthr * 3 * ncnt, sizeof(double));
    double *tled = (double *)calloc((size_t)nthr * LG_N, sizeof(double));
    int64_t *tvis = (int64_t *)calloc((size_t)nthr * ns, sizeof(int64_t));
#pragma omp parallel num_threads(nthr)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double *tABS = tacc + (size_t)tid * 3 * ncnt, *tP = tABS + ncnt, *tLAM = tP + ncnt;
        double *led = ledger ? tled + (size_t)tid * LG_N : NULL;
        int64_t *vis = tvis + (size_t)tid * ns;
        int *sh = (int *)malloc(sizeof(int) * 2 * ns);
        double *ss = (double *)malloc(sizeof(double) * 2 * ns), *mu = (double *)malloc(sizeof(double) * 2 * ns);
        double *phi = (double *)malloc(sizeof(double) * nch), *N = (double *)malloc(sizeof(double) * nch);
#pragma omp for schedule(static, 1)
        for (int i = 0; i < nray; i++) {
            int nseg = ray_path_1d(ns, r, p[i], sh, ss, mu);
            for (int k = 0; k < nsel; k++) {
                int t = sel[k], u = sp->upper[t], l = sp->lower[t];
                double nu = orc_freq(sp, t);
                double kcoef = ORC_C * ORC_C * ORC_C * sp->A[t] / (8.0 * ORC_PI * nu * nu * nu * dv);
                double gr = sp->g[u] / sp->g[l];
                double n0 = bg_photons(nu, tbg, w[i], dv); /* Eq. 1, a = W_i */
                for (int c = 0; c < nch; c++) N[c] = n0;
                if (led) led[LG_INJECTED] += n0 * nch;
                for (int j = 0; j < nseg; j++) {
                    int cell = sh[j];
                    double sig = total_sigma(sp, sigma_turb[cell], tkin[cell]);
                    /* R6: radio convention, v0 = -(v . d) = -v_r mu, mu at the entry of the step */
                    profile_t(sp, t, nch, dv, sig, -vrad[cell] * mu[j], phi);
                    cell_step(nch, N, phi, w[i], ss[j], veff[cell], kcoef, gr, sp->A[t], pops[cell * NL + u],
                              pops[cell * NL + l], ali, &tABS[k * ns + cell], &tP[k * ns + cell], &tLAM[k * ns + cell], led);
                    if (k == 0) vis[cell]++;
                }
                for (int c = 0; c < nch; c++) {
                    if (led) led[LG_ESCAPED] += N[c];
                    if (nout) nout[((size_t)i * nsel + k) * nch + c] = N[c];
                }
            }
        }
        free(sh);
        free(ss);
        free(mu);
        free(phi);
        free(N);
    }
    for (int tid = 0; tid < nthr; tid++) { /* fixed order: thread 0 (rays 0, T, 2T, ...), then thread 1, and so on */
        const double *tABS = tacc + (size_t)tid * 3 * ncnt, *tP = tABS + ncnt, *tLAM = tP + ncnt;
        for (size_t q = 0; q < ncnt; q++) {
            ABS[q] += tABS[q];
            P[q] += tP[q];
            LAM[q] += tLAM[q];
        }
        if (visits)
            for (int c = 0; c < ns; c++) visits[c] += tvis[(size_t)tid * ns + c];
        if (ledger)
            for (int q = 0; q < LG_N; q++) ledger[q] += tled[(size_t)tid * LG_N + q];
    }
    free(tacc);
    free(tled);
    free(tvis);
    free(veff);
    return 0;
}

/* O11 in 1D: spectra T_A(c) for lines of sight at impact parameters b[nlos] */
int orc_spectra_1d(const orc_species *sp, int ns, const double *r, const double *tkin, const double *sigma_turb,
                   const double *vrad, const double *pops, int nch, double band_half, double tbg, int t, int nlos,
                   const double *b, double *TA /* [nlos][nch] */)
{
    int NL = sp->nlevel, u = sp->upper[t], l = sp->lower[t];
    double dv = 2.0 * band_half / nch, nu = orc_freq(sp, t);
    double kcoef = ORC_C * ORC_C * ORC_C * sp->A[t] / (8.0 * ORC_PI * nu * nu * nu * dv);
    double gr = sp->g[u] / sp->g[l];
    double bgI = orc_planck(nu, tbg);
    int *sh = (int *)malloc(sizeof(int) * 2 * ns);
    double *ss = (double *)malloc(sizeof(double) * 2 * ns), *mu = (double *)malloc(sizeof(double) * 2 * ns);
    double *phi = (double *)malloc(sizeof(double) * nch), *I = (double *)malloc(sizeof(double) * nch);
    for (int i = 0; i < nlos; i++) {
        for (int c = 0; c < nch; c++) I[c] = bgI;
        if (b[i] < r[ns - 1]) {
            int nseg = ray_path_1d(ns, r, b[i], sh, ss, mu);
            for (int j = 0; j < nseg; j++) {
                int cell = sh[j];
                double n_u = pops[cell * NL + u], n_l = pops[cell * NL + l];
                double kt = kcoef * (n_l * gr - n_u);
                double Snu = 2.0 * ORC_H * nu * nu * nu / (ORC_C * ORC_C) / (n_l * gr / n_u - 1.0);
                profile_t(sp, t, nch, dv, total_sigma(sp, sigma_turb[cell], tkin[cell]), -vrad[cell] * mu[j], phi);
                for (int c = 0; c < nch; c++) {
                    double tau = kt * phi[c] * ss[j];
                    double ome = -expm1(-tau);
                    I[c] = I[c] * (1.0 - ome) + Snu * ome;
                }
            }
        }
        for (int c = 0; c < nch; c++) TA[(size_t)i * nch + c] = ORC_C * ORC_C / (2.0 * ORC_K * nu * nu) * (I[c] - bgI);
    }
    free(sh);
    free(ss);
    free(mu);
    free(phi);
    free(I);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O8: three-dimensional octree models, readings R7-R11 in DESIGN.md
 *
 * Integer geometry.  Root cell edge = 2^20 units; a level-l cell has edge h_l = 2^(20-l).
 * For a direction d: main axis m = argmax|d| (ties -> lowest index), transverse axes
 * p=(m+1)%3, q=(m+2)%3.  Axes with negative d are mirrored so that in the working frame
 * every ray travels towards +zeta, +x_p, +x_q.  Slopes: S = round_half_even(|d_p/d_m| 2^20);
 * T = floor((2^52 + S/2)/S) (S>0).  The transverse displacement of every ray of the direction is
 *      shift(zeta) = floor(zeta 2^32 / T)        (zeta integer, 0 <= zeta <= N_m 2^20)
 * equivalently the ray crosses transverse offset D>=1 at zeta = ceil(D T / 2^32).
 * Level-k lattice P_k: base positions O + i h_k, O = (25,41)/64 of a root cell (R8).
 * ---------------------------------------------------------------------------------------- */
#define ORC_LB 20
#define ORC_H0 ((int64_t)1 << ORC_LB)

typedef struct {
    int nx, ny, nz;
    int nlev;             /* number of hierarchy levels, >= 1 */
    const int64_t *noff;  /* [nlev+1] offsets of each level in the global cell arrays */
    const int32_t *child; /* [ncell] index (within next level) of first child, -1 = leaf (R17) */
    double root_cm;
} orc_grid;

typedef struct {
    int m, p, q;
    int flip[3];
    uint64_t T[2]; /* p, q; 0 = zero slope */
    double lenf;   /* sqrt(1 + s_p^2 + s_q^2) = 1/|d_m| of the snapped direction */
    double d[3];   /* snapped unit direction, model frame */
    int64_t W[3];  /* extent along m, p, q in units */
} orc_dir;

void orc_setup_dir(const double *din, int nx, int ny, int nz, orc_dir *D)
{
    int n[3] = {nx, ny, nz};
    int m = 0;
    for (int a = 1; a < 3; a++)
        if (fabs(din[a]) > fabs(din[m])) m = a;
    D->m = m;
    D->p = (m + 1) % 3;
    D->q = (m + 2) % 3;
    int ax[3] = {D->m, D->p, D->q};
    double sl[2];
    for (int k = 0; k < 2; k++) {
        double s = fabs(din[ax[k + 1]]) / fabs(din[m]);
        double S = nearbyint(s * 1048576.0); /* round half even (default rounding mode) */
        uint64_t Si = (uint64_t)S;
        if (Si == 0) {
            D->T[k] = 0;
            sl[k] = 0.0;
        } else {
            D->T[k] = (((uint64_t)1 << 52) + Si / 2) / Si;
            sl[k] = 4294967296.0 / (double)D->T[k];
        }
    }
    D->lenf = sqrt(1.0 + sl[0] * sl[0] + sl[1] * sl[1]);
    for (int a = 0; a < 3; a++) D->flip[a] = din[a] < 0.0;
    D->d[m] = (din[m] < 0 ? -1.0 : 1.0) / D->lenf;
    D->d[D->p] = (din[D->p] < 0 ? -1.0 : 1.0) * sl[0] / D->lenf;
    D->d[D->q] = (din[D->q] < 0 ? -1.0 : 1.0) * sl[1] / D->lenf;
    for (int k = 0; k < 3; k++) D->W[k] = (int64_t)n[ax[k]] * ORC_H0;
}

static inline int64_t shift_of(uint64_t T, int64_t zeta)
{
    if (T == 0) return 0;
    return (int64_t)((((unsigned __int128)(uint64_t)zeta) << 32) / T);
}
/* smallest zeta with shift(zeta) >= D */
static inline int64_t cross_of(uint64_t T, int64_t D)
{
    if (D <= 0) return 0;
    if (T == 0) return INT64_MAX;
    unsigned __int128 v = (unsigned __int128)(uint64_t)D * T;
    return (int64_t)((v + (((unsigned __int128)1 << 32) - 1)) >> 32);
}

typedef struct {
    int64_t cell[16]; /* global index of the ancestor at each level up to the leaf */
    int level;
    int64_t org[3]; /* lower corner of the leaf in the working frame (zeta, xp, xq) */
    int64_t h;
} orc_leaf;

/* leaf containing the integer point f = (zeta, xp, xq) of the working frame */
static void find_leaf(const orc_grid *G, const orc_dir *D, const int64_t *f, orc_leaf *L)
{
    int64_t X[3];
    int ax[3] = {D->m, D->p, D->q};
    for (int k = 0; k < 3; k++) X[ax[k]] = D->flip[ax[k]] ? D->W[k] - 1 - f[k] : f[k];
    int64_t ix = X[0] >> ORC_LB, iy = X[1] >> ORC_LB, iz = X[2] >> ORC_LB;
    int64_t g = G->noff[0] + ix + (int64_t)G->nx * (iy + (int64_t)G->ny * iz);
    int l = 0;
    L->cell[0] = g;
    while (G->child[g] >= 0) {
        int bit = ORC_LB - 1 - l;
        int cx = (int)((X[0] >> bit) & 1), cy = (int)((X[1] >> bit) & 1), cz = (int)((X[2] >> bit) & 1);
        g = G->noff[l + 1] + G->child[g] + cx + 2 * cy + 4 * cz;
        l++;
        L->cell[l] = g;
    }
    L->level = l;
    L->h = ORC_H0 >> l;
    for (int k = 0; k < 3; k++) L->org[k] = f[k] & ~(L->h - 1);
}

typedef struct {
    const orc_species *sp;
    const orc_grid *G;
    const double *tkin, *sigma_turb, *vx, *vy, *vz, *pops;
    int nch;
    double dv, tbg;
    int ndir, nsel;
    const int *sel;
    int ali, geom_only;
    double *ABS, *P, *LAM;
    int64_t *visits, *pathz;
    double **dspec; /* donor intensity per refined cell: [nsel][nch], N/a */
    int64_t ncell;
} sim3_ctx;

/* Trace one line of the level-`tag` lattice with base (bp,bq) through the whole model (O8).
 * Steps are taken in every leaf (alive or not); radiative work only where level >= tag.          */
static void trace_line(const sim3_ctx *S, const orc_dir *D, int tag, int64_t bp, int64_t bq, double *N /*[nsel][nch]*/,
                       double *phi, double *ledger)
{
    const orc_species *sp = S->sp;
    const orc_grid *G = S->G;
    int NL = sp->nlevel, nch = S->nch, nsel = S->nsel;
    int64_t zend = D->W[0];
    double u_cm = G->root_cm / (double)ORC_H0;
    int alive = 0;
    double a_cur = 0.0;
    int64_t zeta = 0;
    int64_t wrap_prev[2] = {0, 0};
    int first = 1;
    while (zeta < zend) {
        int64_t up = bp + shift_of(D->T[0], zeta), uq = bq + shift_of(D->T[1], zeta);
        int64_t wr[2] = {up / D->W[1], uq / D->W[2]};
        int64_t f[3] = {zeta, up % D->W[1], uq % D->W[2]};
        orc_leaf L;
        find_leaf(G, D, f, &L);
        int wrapped = !first && (wr[0] != wrap_prev[0] || wr[1] != wrap_prev[1]);
        wrap_prev[0] = wr[0];
        wrap_prev[1] = wr[1];
        double hcm = G->root_cm / (double)(1 << L.level);
        double a_new = hcm * hcm / (D->lenf * S->ndir); /* a = h^2 |d_m| / NDIR (O5) */
        int can_live = L.level >= tag;
        if (!S->geom_only) {
            /* ---- state change on entering leaf L (O8: alive / birth / termination / wrap) ---- */
            if (alive) {
                if (wrapped) { /* leaves through a side: photons escape; new ray on the opposite side */
                    for (int i = 0; i < nsel * nch; i++) ledger[LG_ESCAPED] += N[i];
                    alive = 0;
                } else if (can_live) { /* intensity continuous, photons rescaled with a */
                    double fsc = a_new / a_cur;
                    if (fsc != 1.0)
                        for (int i = 0; i < nsel * nch; i++) {
                            ledger[LG_RESCALE] += N[i] * (1.0 - fsc);
                            N[i] *= fsc;
                        }
                } else { /* entering a region refined to less than the tag: terminated */
                    for (int i = 0; i < nsel * nch; i++) ledger[LG_TERMINATED] += N[i];
                    alive = 0;
                }
            }
            if (!alive && can_live) {
                if (first || wrapped) { /* model boundary: background, Eq. 1 */
                    for (int k = 0; k < nsel; k++) {
                        double n0 = bg_photons(orc_freq(sp, S->sel[k]), S->tbg, a_new, S->dv);
                        for (int c = 0; c < nch; c++) N[k * nch + c] = n0;
                        ledger[LG_INJECTED] += n0 * nch;
                    }
                } else { /* birth at an interior face: intensity of the donor of the level-(tag-1) ancestor */
                    const double *ds = S->dspec[L.cell[tag - 1]];
                    for (int i = 0; i < nsel * nch; i++) {
                        N[i] = ds[i] * a_new;
                        ledger[LG_CREATED] += N[i];
                    }
                }
                alive = 1;
            }
            a_cur = a_new;
            /* ---- donor duty: store intensity at the upstream face of every refined ancestor entered now ---- */
            if (alive)
                for (int j = tag; j < L.level; j++)
                    if ((zeta & ((ORC_H0 >> j) - 1)) == 0) {
                        double *ds = S->dspec[L.cell[j]];
                        if (!ds) {
                            ds = (double *)malloc(sizeof(double) * nsel * nch);
                            S->dspec[L.cell[j]] = ds;
                        }
                        for (int i = 0; i < nsel * nch; i++) ds[i] = N[i] / a_cur;
                    }
        } else {
            alive = can_live;
        }
        /* ---- next event: first zeta at which the point leaves the leaf ---- */
        int64_t zmain = L.org[0] + L.h;
        int64_t zp = cross_of(D->T[0], L.org[1] + L.h - f[1] + shift_of(D->T[0], zeta));
        int64_t zq = cross_of(D->T[1], L.org[2] + L.h - f[2] + shift_of(D->T[1], zeta));
        int64_t znext = zmain;
        if (zp < znext) znext = zp;
        if (zq < znext) znext = zq;
        int64_t dz = znext - zeta;
        if (alive) {
            int64_t cell = L.cell[L.level];
#pragma omp atomic
            S->visits[cell]++;
#pragma omp atomic
            S->pathz[cell] += dz;
            if (!S->geom_only) {
                double s = (double)dz * u_cm * D->lenf;
                double veff = hcm * hcm * hcm;
                double v0 = -(S->vx[cell] * D->d[0] + S->vy[cell] * D->d[1] + S->vz[cell] * D->d[2]); /* R6 */
                for (int k = 0; k < nsel; k++) {
                    int t = S->sel[k], u = sp->upper[t], l = sp->lower[t];
                    double nu = orc_freq(sp, t);
                    profile_t(sp, t, nch, S->dv, total_sigma(sp, S->sigma_turb[cell], S->tkin[cell]), v0, phi);
                    double kcoef = ORC_C * ORC_C * ORC_C * sp->A[t] / (8.0 * ORC_PI * nu * nu * nu * S->dv);
                    cell_step(nch, N + k * nch, phi, a_cur, s, veff, kcoef, sp->g[u] / sp->g[l], sp->A[t],
                              S->pops[cell * NL + u], S->pops[cell * NL + l], S->ali, &S->ABS[(size_t)k * S->ncell + cell],
                              &S->P[(size_t)k * S->ncell + cell], &S->LAM[(size_t)k * S->ncell + cell], ledger);
                }
            }
        }
        zeta = znext;
        first = 0;
    }
    if (alive && !S->geom_only)
        for (int i = 0; i < nsel * nch; i++) ledger[LG_ESCAPED] += N[i];
}

/* O5-O8 simulation over all directions.  Outputs ABS,P,LAM [nsel][ncell]; visits,pathz [ncell]; ledger[LG_N].
 * Passes by tag: lines of P_0 first, then tag 1, ... so that every donor spectrum exists before it is needed. */
int orc_sim_3d(const orc_species *sp, const orc_grid *G, const double *tkin, const double *sigma_turb, const double *vx,
               const double *vy, const double *vz, const double *pops, int nch, double band_half, double tbg, int ndir,
               const double *dirs, int nsel, const int *sel, int ali, int geom_only, const int *off64 /* lattice offset in 1/64 root cell: {25,41} (R8) */,
               double *ABS, double *P, double *LAM, int64_t *visits, int64_t *pathz, double *ledger,
               int root_stride /* > 1: TIMING SAMPLE ONLY (bench.py): every root_stride-th line of the root lattice, no finer lattices */)
{
    int64_t ncell = G->noff[G->nlev];
    sim3_ctx S;
    S.sp = sp; S.G = G; S.tkin = tkin; S.sigma_turb = sigma_turb; S.vx = vx; S.vy = vy; S.vz = vz; S.pops = pops;
    S.nch = nch; S.dv = 2.0 * band_half / nch; S.tbg = tbg; S.ndir = ndir; S.nsel = nsel; S.sel = sel; S.ali = ali;
    S.geom_only = geom_only; S.ABS = ABS; S.P = P; S.LAM = LAM; S.visits = visits; S.pathz = pathz; S.ncell = ncell;
    S.dspec = (double **)calloc((size_t)ncell, sizeof(double *));
    if (!geom_only) {
        memset(ABS, 0, sizeof(double) * nsel * ncell);
        memset(P, 0, sizeof(double) * nsel * ncell);
        memset(LAM, 0, sizeof(double) * nsel * ncell);
    }
    memset(visits, 0, sizeof(int64_t) * ncell);
    memset(pathz, 0, sizeof(int64_t) * ncell);
    double led[LG_N];
    memset(led, 0, sizeof(led));
    for (int id = 0; id < ndir; id++) {
        orc_dir D;
        orc_setup_dir(dirs + 3 * id, G->nx, G->ny, G->nz, &D);
        for (int tag = 0; tag < (root_stride > 1 ? 1 : G->nlev); tag++) {
            int64_t hk = ORC_H0 >> tag;
            int64_t np = D.W[1] / hk, nq = D.W[2] / hk;
            int64_t Op = off64[0] * (ORC_H0 / 64), Oq = off64[1] * (ORC_H0 / 64);
#pragma omp parallel
            {
                double *N = (double *)malloc(sizeof(double) * (nsel > 0 ? nsel : 1) * nch);
                double *phi = (double *)malloc(sizeof(double) * nch);
                double lled[LG_N];
                memset(lled, 0, sizeof(lled));
#pragma omp for schedule(dynamic, 16)
                for (int64_t ij = 0; ij < np * nq; ij++) {
                    int64_t i = ij % np, j = ij / np;
                    if (tag > 0 && !((i & 1) || (j & 1))) continue; /* belongs to a coarser lattice */
                    if (root_stride > 1 && ij % root_stride) continue; /* bounded sample of the rays (no result is used) */
                    trace_line(&S, &D, tag, Op + i * hk, Oq + j * hk, N, phi, lled);
                }
#pragma omp critical
                for (int k = 0; k < LG_N; k++) led[k] += lled[k];
                free(N);
                free(phi);
            }
        }
        for (int64_t c = 0; c < ncell; c++)
            if (S.dspec[c]) {
                free(S.dspec[c]);
                S.dspec[c] = NULL;
            }
    }
    free(S.dspec);
    if (ledger) memcpy(ledger, led, sizeof(led));
    return 0;
}

/* Per-leaf count of crossing lines and of the main-axis path for one direction, computed one leaf at
 * a time from the lattice definition alone (used to sample full-size models).  leaf_org is the lower
 * corner of the leaf in MODEL integer coordinates, level its level.                                   */
void orc_leaf_visits(const orc_grid *G, const double *dir, const int64_t *leaf_org_model, int level, int64_t *nvisit,
                     int64_t *pathz)
{
    orc_dir D;
    orc_setup_dir(dir, G->nx, G->ny, G->nz, &D);
    int ax[3] = {D.m, D.p, D.q};
    int64_t h = ORC_H0 >> level, org[3];
    for (int k = 0; k < 3; k++) {
        int64_t lo = leaf_org_model[ax[k]];
        org[k] = D.flip[ax[k]] ? D.W[k] - (lo + h) : lo;
    }
    int64_t Op = 25 * (ORC_H0 / 64), Oq = 41 * (ORC_H0 / 64);
    int64_t nv = 0, pz = 0;
    /* Lines of P_level: base O + i*h, i any integer (negative i = images that wrapped around).  A line
     * can only cross the leaf if at zeta = org[0] it lies within one cell edge below the leaf (slopes <= 1);
     * the candidate range below is generous and every candidate is tested exactly.                        */
    int64_t ip0 = (org[1] - Op - shift_of(D.T[0], org[0]) - 3 * h) / h - 2;
    int64_t iq0 = (org[2] - Oq - shift_of(D.T[1], org[0]) - 3 * h) / h - 2;
    for (int64_t i = ip0; i < ip0 + 10; i++)
        for (int64_t j = iq0; j < iq0 + 10; j++) {
            int64_t bp = Op + i * h, bq = Oq + j * h;
            if (bp >= D.W[1] || bq >= D.W[2]) continue; /* not a line of the model */
            int64_t zin = org[0], zout = org[0] + h, z;
            z = cross_of(D.T[0], org[1] - bp); if (z > zin) zin = z;
            z = cross_of(D.T[1], org[2] - bq); if (z > zin) zin = z;
            z = cross_of(D.T[0], org[1] + h - bp); if (z < zout) zout = z;
            z = cross_of(D.T[1], org[2] + h - bq); if (z < zout) zout = z;
            if (zout > zin) {
                nv++;
                pz += zout - zin;
            }
        }
    *nvisit = nv;
    *pathz = pz;
}

/* position of a lattice line at zeta (working frame), for the brute-force geometry pin P9 */
void orc_line_position(const double *dir, int nx, int ny, int nz, int64_t bp, int64_t bq, int64_t zeta, int64_t *xp,
                       int64_t *xq)
{
    orc_dir D;
    orc_setup_dir(dir, nx, ny, nz, &D);
    *xp = bp + shift_of(D.T[0], zeta);
    *xq = bq + shift_of(D.T[1], zeta);
}

/* O11: spectral map.  One straight line of sight per pixel along `dir`, through all leaves, no births.
 * Pixel (ix,iy) starts at zeta=0 at the working-frame transverse position given by the integer affine map `aff`
 * (supplied by the caller); the line ends when it leaves the model through any face.  T_A in K.          */
int orc_spectra_3d(const orc_species *sp, const orc_grid *G, const double *tkin, const double *sigma_turb, const double *vx,
                   const double *vy, const double *vz, const double *pops, int nch, double band_half, double tbg, int t,
                   const double *dir, int npx, int npy, const int64_t *aff /* x0p,x0q, dpx/dix,dpx/diy, dqx/dix,dqx/diy */,
                   double *TA /*[npy][npx][nch]*/)
{
    orc_dir D;
    orc_setup_dir(dir, G->nx, G->ny, G->nz, &D);
    int NL = sp->nlevel, u = sp->upper[t], l = sp->lower[t];
    double dv = 2.0 * band_half / nch, nu = orc_freq(sp, t);
    double kcoef = ORC_C * ORC_C * ORC_C * sp->A[t] / (8.0 * ORC_PI * nu * nu * nu * dv);
    double gr = sp->g[u] / sp->g[l], bgI = orc_planck(nu, tbg), u_cm = G->root_cm / (double)ORC_H0;
#pragma omp parallel
    {
        double *phi = (double *)malloc(sizeof(double) * nch), *I = (double *)malloc(sizeof(double) * nch);
#pragma omp for schedule(dynamic, 8)
        for (int64_t pxy = 0; pxy < (int64_t)npx * npy; pxy++) {
            int ix = (int)(pxy % npx), iy = (int)(pxy / npx);
            int64_t bp = aff[0] + ix * aff[2] + iy * aff[3], bq = aff[1] + ix * aff[4] + iy * aff[5];
            for (int c = 0; c < nch; c++) I[c] = bgI;
            int64_t zeta = 0;
            /* advance to the first zeta at which the point is inside the transverse extent (entry through a side) */
            if (bp < 0) { int64_t z = cross_of(D.T[0], -bp); if (z > zeta) zeta = z; }
            if (bq < 0) { int64_t z = cross_of(D.T[1], -bq); if (z > zeta) zeta = z; }
            while (zeta < D.W[0]) {
                int64_t up = bp + shift_of(D.T[0], zeta), uq = bq + shift_of(D.T[1], zeta);
                if (up < 0 || uq < 0 || up >= D.W[1] || uq >= D.W[2]) break;
                int64_t f[3] = {zeta, up, uq};
                orc_leaf L;
                find_leaf(G, &D, f, &L);
                int64_t znext = L.org[0] + L.h, z;
                z = cross_of(D.T[0], L.org[1] + L.h - bp); if (z < znext) znext = z;
                z = cross_of(D.T[1], L.org[2] + L.h - bq); if (z < znext) znext = z;
                int64_t cell = L.cell[L.level];
                double s = (double)(znext - zeta) * u_cm * D.lenf;
                double n_u = pops[cell * NL + u], n_l = pops[cell * NL + l];
                double kt = kcoef * (n_l * gr - n_u);
                double Snu = 2.0 * ORC_H * nu * nu * nu / (ORC_C * ORC_C) / (n_l * gr / n_u - 1.0);
                double v0 = -(vx[cell] * D.d[0] + vy[cell] * D.d[1] + vz[cell] * D.d[2]);
                profile_t(sp, t, nch, dv, total_sigma(sp, sigma_turb[cell], tkin[cell]), v0, phi);
                for (int c = 0; c < nch; c++) {
                    double ome = -expm1(-kt * phi[c] * s);
                    I[c] = I[c] * (1.0 - ome) + Snu * ome;
                }
                zeta = znext;
            }
            for (int c = 0; c < nch; c++)
                TA[((size_t)iy * npx + ix) * nch + c] = ORC_C * ORC_C / (2.0 * ORC_K * nu * nu) * (I[c] - bgI);
        }
        free(phi);
        free(I);
    }
    return 0;
}

/* Standalone cell-step sequence on one ray (pins P1, P2): nstep steps with given s, phi shared. */
void orc_slab(const orc_species *sp, int t, int nch, double band_half, double tbg, double a, double veff_each, int nstep,
              const double *s, double sigma, double v0, double n_u, double n_l, int ali, double *N /* in/out [nch] */,
              double *acc /* ABS,P,LAM sums */, double *ledger, int inject)
{
    double dv = 2.0 * band_half / nch, nu = orc_freq(sp, t);
    double kcoef = ORC_C * ORC_C * ORC_C * sp->A[t] / (8.0 * ORC_PI * nu * nu * nu * dv);
    double *phi = (double *)malloc(sizeof(double) * nch);
    profile_t(sp, t, nch, dv, sigma, v0, phi);
    if (inject)
        for (int c = 0; c < nch; c++) N[c] = bg_photons(nu, tbg, a, dv);
    acc[0] = acc[1] = acc[2] = 0.0;
    for (int j = 0; j < nstep; j++)
        cell_step(nch, N, phi, a, s[j], veff_each, kcoef, sp->g[sp->upper[t]] / sp->g[sp->lower[t]], sp->A[t], n_u, n_l, ali,
                  &acc[0], &acc[1], &acc[2], ledger);
    free(phi);
}

void orc_profile(int nch, double dv, double sigma, double v0, double *phi) { profile(nch, dv, sigma, v0, phi); }
void orc_profile_t(const orc_species *sp, int t, int nch, double dv, double sigma, double v0, double *phi) { profile_t(sp, t, nch, dv, sigma, v0, phi); }
