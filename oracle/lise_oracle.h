/*
 * lise_oracle.h -- CPU oracle for the TDSLDA hot path of arxiv/paper_2009_00745 (the LISE package).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or constant generator with the CUDA library (paper_2009_00745_b200/csrc, include/lise.h).
 *
 * Plain C11, fp64 (complex128), slow on purpose: every spatial derivative is the lattice operator
 * F^-1 (ik)^m F of PAPER.md Eqs. 49-50 written out as a dense N x N matrix built term by term from
 * the DFT sums of Eq. 49 (no FFT anywhere), every formula follows SURVEY.md Appendix A (the adopted
 * reading of PAPER.md Eqs. 3, 9, 11-21, 43-44, 49-51, 55, 56, 58-62, 75-78, 80-81).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md section "Oracle pins".
 * Parity unpinned (parameters only, no formula): Skyrme parameter values, g0, alpha = 0, the
 * details of the series-expansion starter (readings B14, B16, B18).
 *
 * All pointers are HOST pointers.  Wavefunction block layout:
 *   [state][component: u_up, u_dn, v_up, v_dn][ix][iy][iz], iz fastest, interleaved complex128.
 * Species 0 = neutrons, 1 = protons.  All calls return 0 on success, negative on error.
 */
#ifndef LISE_ORACLE_H
#define LISE_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lise_ref_ctx lise_ref_ctx;

typedef struct {
    double hbar2_2m, e2, hbarc;                      /* MeV fm^2, MeV fm, MeV fm */
    double t0, t1, t2, t3, x0, x1, x2, x3, gamma, W0; /* Skyrme set (default SLy4) */
    double g0_n, g0_p;                               /* bare pairing couplings, MeV fm^3; 0 = off */
    int coulomb, pairing_rearrangement, remove_phase;
    /* functional and pairing variants (Eqs. 8, 10, 15, 20; defaults: all off / zero) */
    double alpha_pair;                               /* Eq. 8: g0(r) = g0 (1 - alpha n(r) / n0), n = n_n + n_p, n0 = 0.16 fm^-3 */
    double mu_n, mu_p, e_cut;                        /* Eq. 20: chemical potentials and energy cutoff E_c (MeV), spherical cutoff */
    double sea_a[3], sea_b[3], sea_c[3];             /* Eq. 10: SeaLL1 volume coefficients a_j, b_j, c_j (ref. [36]: not printed) */
    double sea_cdn[2], sea_cdj[2];                   /* SeaLL1: C_t^{n Delta n}, C_t^{nabla J}, t = 0, 1 */
    int functional;                                  /* 0 Skyrme (Eq. 9), 1 SeaLL1 (Eq. 10) */
    int pairing_cutoff;                              /* 0 lattice cutoff (Eq. 21), 1 spherical cutoff (Eq. 20) */
    int renormalize;                                 /* 1: every qpwf is normalised at the end of each step (L637) */
} lise_ref_params;

/* Eqs. 37-41 and the energy of the external terms; coordinates x_i = i dx (Eq. 43), Q_lm about the total c.m. */
typedef struct {
    double rcm[3], rcm_n[3], rcm_p[3];               /* Eq. 37, fm */
    double q20, q30, q40, q21[2], q22[2];            /* Eq. 38 b-e of the total density (re, im for m != 0) */
    double delta_n, delta_p;                         /* Eq. 39, MeV */
    double e_coll;                                   /* Eq. 40 read as sum_q int (hbar^2/2m) j_q^2 / n_q, MeV */
    double v_cm[3], e_cm;                            /* Eqs. 27, 41: units of c; MeV */
    double e_ext;                                    /* expectation value of the external terms of Eqs. 24, 26, 36, MeV */
} lise_ref_observables_ext_t;

typedef struct {
    double energy, e_kin, e_skyrme, e_coul, e_pair;
    double n_neutron, n_proton;
    double norm_defect;   /* max_k | <psi_k|psi_k> - 1 |                                          */
    double ortho_defect;  /* max over pairs (k, (k+d) mod nwf), d in {1, 2, nwf/2}, of |<k|l>|     */
    double time;          /* fm/c */
    long step;
} lise_ref_observables_t;

int  lise_ref_default_params(lise_ref_params *p);
int  lise_ref_create(int nx, int ny, int nz, double dx, double dt, int nwf_n, int nwf_p, lise_ref_ctx **out);
void lise_ref_destroy(lise_ref_ctx *c);
int  lise_ref_set_params(lise_ref_ctx *c, const lise_ref_params *p);
int  lise_ref_set_dt(lise_ref_ctx *c, double dt);                 /* resets the multistep history */
int  lise_ref_set_num_threads(int n);                             /* OpenMP threads; returns count in use */
int  lise_ref_set_wavefunctions(lise_ref_ctx *c, int species, const void *psi);
int  lise_ref_get_wavefunctions(lise_ref_ctx *c, int species, void *psi);
int  lise_ref_densities(lise_ref_ctx *c, int species, double *out14);   /* Table 2 layout, 14*Nxyz */
int  lise_ref_potentials(lise_ref_ctx *c, int species, double *out14);  /* Table 3 rows 0..13: U, M, lap M, W, S, A, Delta */
int  lise_ref_apply_h(lise_ref_ctx *c, int species, const void *in, void *out, int nstates);
int  lise_ref_step(lise_ref_ctx *c, int nsteps);
int  lise_ref_observables(lise_ref_ctx *c, lise_ref_observables_t *out);

/* ---- finer-grained entry points used by the pin tests ---- */
/* dense lattice derivative matrix of one axis, order 1 (Nyquist zeroed) or 2; out is N*N doubles, row-major */
int  lise_ref_deriv_matrix(lise_ref_ctx *c, int axis, int order, double *out);
/* apply D_axis (order 1) or D2_axis (order 2) to nfields complex fields of Nxyz points */
int  lise_ref_deriv(lise_ref_ctx *c, int axis, int order, const void *in, void *out, int nfields);
/* Coulomb potential of a real density (Eqs. 58-62, padded cube of side 3*max(N)); phi is Nxyz doubles */
int  lise_ref_coulomb(lise_ref_ctx *c, const double *n_p, double *phi);
/* potentials and energy from externally supplied Table-2 densities (both species); pot_* are 14*Nxyz, e5 = {E, kin, skyrme, coul, pair} */
int  lise_ref_potentials_from(lise_ref_ctx *c, const double *dens_n, const double *dens_p,
                              double *pot_n, double *pot_p, double *e5);
/* H psi with externally supplied Table-3 potentials of that species */
int  lise_ref_apply_h_with(lise_ref_ctx *c, const double *pot14, const void *in, void *out, int nstates);
/* Table-2 densities of an arbitrary block of states (not the context's) */
int  lise_ref_densities_of(lise_ref_ctx *c, const void *psi, int nstates, double *out14);
/* the two halves of Eq. 78 on flat complex arrays of n elements (exactly the routines lise_ref_step uses) */
int  lise_ref_abm_predict(long n, double dt, const void *y_n, const void *y_nm1,
                          const void *f_n, const void *f_nm1, const void *f_nm2, const void *f_nm3,
                          const void *e_n, void *p_out, void *m_out);
int  lise_ref_abm_correct(long n, double dt, const void *y_n, const void *y_nm1,
                          const void *fm, const void *f_n, const void *f_nm1, const void *f_nm2,
                          const void *p, void *y_out, void *e_out);
/* overwrite the multistep history of one species and mark the context as started (step counter >= 3) */
int  lise_ref_set_history(lise_ref_ctx *c, int species, const void *y_nm1,
                          const void *f_nm1, const void *f_nm2, const void *f_nm3, const void *e_n);
/* ---- (f)2: restart (L764-L768), (f)4: boosts, external fields, moving / rotating frame (Eqs. 23-36) ---- */
/* sets the clock and the total step counter; the multistep start-up state is not touched (after
 * lise_ref_set_wavefunctions the next three steps use the starter: that is the restart of L764-L768) */
int  lise_ref_set_time(lise_ref_ctx *c, double time, long step);
/* Eq. 23: u -> e^{i chi} u, v -> e^{-i chi} v for every state of the species (chi: Nxyz doubles); restarts the multistep method */
int  lise_ref_boost(lise_ref_ctx *c, int species, const double *chi);
/* Eq. 24: h_q -> h_q + U0 - (1/2) [Uvec . p + p . Uvec]; u0: Nxyz doubles (MeV), uvec: 3 Nxyz doubles (units of c); NULL = none */
int  lise_ref_set_external_fields(lise_ref_ctx *c, int species, const double *u0, const double *uvec);
/* L232: the fields of Eq. 24 depend on time.  The stored profiles are multiplied by f_now wherever H is built from y_n
 * (time t_n: first evaluation of Eq. 78, Eq. 75, potentials / apply_h / observables of the current state), by f_next in
 * the evaluation on the modifier (time t_{n+1}, Eq. 78c), and by (f_now + f_next) / 2 in the starter's H_cor, whose
 * densities are averaged the same way (Eq. 76; reading B33).  Default 1, 1.  Frame terms are not scaled.
 * The pair holds until it is set again: a driven run calls this before every single step. */
int  lise_ref_set_external_amplitudes(lise_ref_ctx *c, double f_now, double f_next);
/* Eqs. 26, 36: h -> h - v_cm . p - omega . (l + s), l = (r - origin) x p; v_cm in units of c, omega in c / fm, origin in fm */
int  lise_ref_set_frame(lise_ref_ctx *c, const double *v_cm, const double *omega, const double *origin);
/* Eqs. 37-41 of the current wavefunctions / of externally supplied Table-2 densities and Table-3 potentials */
int  lise_ref_observables_ext(lise_ref_ctx *c, lise_ref_observables_ext_t *out);
int  lise_ref_moments_from(lise_ref_ctx *c, const double *dens_n, const double *dens_p,
                           const double *pot_n, const double *pot_p, lise_ref_observables_ext_t *out);
/* 1 / g_eff of Eq. 20a for one point (M = hbar^2 / 2 m*, U, mu, E_c in MeV; g0 in MeV fm^3): the pin tests' entry */
double lise_ref_inv_geff_spherical(double g0, double M, double U, double mu, double e_cut);
/* pairing constant K of Eq. 21 as the oracle uses it */
double lise_ref_pairing_K(void);

#ifdef __cplusplus
}
#endif
#endif
