/*
 * lise.h -- C-ABI boundary of the B200-native TDSLDA time-step library (liblise.so).
 *
 * One thing is built here: the data-parallel hot path of arxiv/paper_2009_00745 (the LISE package) --
 * the TDSLDA right-hand side and the Adams-Bashforth-Milne (ABM) step applied to every quasiparticle
 * wavefunction (qpwf) on a periodic 3D lattice.  All arithmetic is IEEE fp64 (complex128) in
 * hand-written CUDA kernels for sm_100a; there is no CPU fallback and no cuFFT/cuBLAS on this path.
 * Citations are "PAPER.md:L<line>" of the paper text plus equation numbers; the adopted reading of
 * every garbled or ambiguous passage is listed in DESIGN.md (ledger B1..B32).
 *
 * Conventions
 *   species     0 = neutrons, 1 = protons; nwf_p = 0 means this context holds no proton states: Coulomb then defaults
 *               to off (a state-sharded rank without protons switches it on with lise_set_params, see below).
 *   lattice     nx, ny, nz even; lattice constant dx = dy = dz (Eq. 43); volume element dV = dx^3.
 *   wavefunction block ("psi"): [state][component: u_up, u_dn, v_up, v_dn][ix][iy][iz], iz fastest,
 *               interleaved (re, im) doubles (Eq. 1; the order inside xyz is this library's choice).
 *               States are normalised as dV * sum |psi|^2 = 1, so densities are in fm^-3.
 *   pointers    every `*_dev` argument is a DEVICE pointer owned by the caller (e.g. a torch tensor);
 *               the library reads/writes it on the context's stream and never frees or retains it.
 *               Every other pointer is a HOST pointer.
 *   ordering    calls enqueue work on the context's stream and return without synchronising, except
 *               lise_observables (synchronises, writes host memory) and lise_create / lise_destroy.
 *   errors      every call returns LISE_OK (0) or a negative LISE_E* code; nothing throws or aborts.
 *               lise_last_error(ctx) gives a human-readable message for the last failure (ctx = NULL: for the
 *               calling thread's last failed lise_create).  The library prints nothing.
 *   units       MeV, fm, fm/c.
 */
#ifndef LISE_H
#define LISE_H

#ifdef __cplusplus
extern "C" {
#endif

enum {
    LISE_OK = 0,
    LISE_EINVAL = -1,       /* bad argument (null pointer, odd lattice size, species out of range ...) */
    LISE_ESTATE = -2,       /* call order: wavefunctions of a species not set yet                      */
    LISE_ECUDA = -3,        /* a CUDA runtime call or kernel launch failed                             */
    LISE_ENOMEM = -4,       /* device memory allocation failed                                         */
    LISE_EUNSUPPORTED = -5  /* lattice too large for the on-chip plane tiles of this build             */
};

typedef struct lise_ctx lise_ctx; /* opaque; owns every internal device buffer */

/* Physical parameters.  None is printed in the paper; defaults (lise_default_params) are SLy4
 * (the paper's default force) and volume pairing with the cubic-cutoff
 * renormalisation of Eq. 21. */
typedef struct {
    double hbar2_2m, e2, hbarc;                         /* 20.73553 MeV fm^2, 1.439964 MeV fm, 197.3269804 MeV fm */
    double t0, t1, t2, t3, x0, x1, x2, x3, gamma, W0;   /* Skyrme parameters -> couplings of Eq. 9               */
    double g0_n, g0_p;                                  /* bare pairing couplings, MeV fm^3 (0 = pairing off)    */
    int coulomb;                                        /* 1: Coulomb direct (Eqs. 58-62) + Slater exchange (Eq. 6) for protons; the flag
                                                         * alone decides (it must be the same on every rank of a state-sharded run) */
    int pairing_rearrangement;                          /* 1: include d E_pair / d n in U (reading B8) */
    int remove_phase;                                   /* 1: subtract eta_k = <psi_k|H|psi_k> (Eqs. 80-81)      */
    /* functional and pairing variants; lise_default_params leaves them off / zero */
    double alpha_pair;                                  /* Eq. 8: g0(r) = g0 (1 - alpha n(r) / n0), n = n_n + n_p, n0 = 0.16 fm^-3:
                                                         * 0 volume, 1 surface, 1/2 mixed pairing                              */
    double mu_n, mu_p, e_cut;                           /* Eq. 20: chemical potentials and energy cutoff E_c (MeV) of the
                                                         * spherical-cutoff renormalisation (used when pairing_cutoff = 1)   */
    double sea_a[3], sea_b[3], sea_c[3];                /* Eq. 10: SeaLL1 volume coefficients a_j, b_j, c_j, j = 0..2 (values of
                                                         * ref. [36], not printed in the paper: supplied by the caller)      */
    double sea_cdn[2], sea_cdj[2];                      /* SeaLL1: C_t^{n Delta n} and C_t^{nabla J}, t = 0, 1                */
    int functional;                                     /* 0: Skyrme functional (Eq. 9); 1: SeaLL1 (Eqs. 10, 15; m* = m)     */
    int pairing_cutoff;                                 /* 0: lattice cutoff, Eq. 21; 1: spherical cutoff, Eq. 20 (no pairing
                                                         * rearrangement term then: DESIGN.md reading B30)                   */
    int renormalize;                                    /* 1: every qpwf is normalised at the end of each step */
} lise_params;

/* Observables of PAPER.md Eqs. 37-41 (L304-L335) of the current wavefunctions y_n, and the energy of the external
 * terms.  Coordinates are x_i = i dx (Eq. 43); the multipoles are taken about the total centre of mass (L367). */
typedef struct {
    double rcm[3], rcm_n[3], rcm_p[3];                  /* Eq. 37: centre of mass of nucleons, neutrons, protons, fm            */
    double q20, q30, q40, q21[2], q22[2];               /* Eq. 38 b-e of the total density: 2z^2-x^2-y^2, z(2z^2-3x^2-3y^2),
                                                         * 35z^4-30z^2r^2+3r^4, (x+iy)z and (x+iy)^2 as (re, im)               */
    double delta_n, delta_p;                            /* Eq. 39: density-weighted average of |Delta_q|, MeV                   */
    double e_coll;                                      /* Eq. 40 read as sum_q int (hbar^2/2m) j_q^2 / n_q (B31), MeV */
    double v_cm[3], e_cm;                               /* Eqs. 27, 41: hbar int j / (m A) in units of c; (1/2) m A v_cm^2, MeV  */
    double e_ext;                                       /* expectation value of the external terms (Eqs. 24, 26, 36), MeV       */
} lise_observables_ext_t;

/* Observables of the current wavefunctions y_n (E(t), Z(t), N(t)). */
typedef struct {
    double energy, e_kin, e_skyrme, e_coul, e_pair;     /* Eq. 4 and its parts (Eqs. 5-9), MeV               */
    double n_neutron, n_proton;                         /* dV * sum n_q                                      */
    double norm_defect;                                 /* max_k | <psi_k|psi_k> - 1 |                       */
    double ortho_defect;                                /* max over pairs (k, (k+d) mod nwf), d in {1, 2, nwf/2}, of |<psi_k|psi_l>| */
    double time;                                        /* fm/c                                              */
    long step;                                          /* steps taken since the last lise_set_wavefunctions */
} lise_observables_t;

int lise_default_params(lise_params *p);

/* Allocates a context for an nx x ny x nz lattice with spacing dx (fm), time step dt (fm/c) and
 * nwf_n / nwf_p quasiparticle states.  Device memory: 7 state arrays per species
 * (y_n, y_{n-1}, three f = dy/dt history arrays, e_n = p_n - c_n, predictor scratch; the paper's
 * code holds 11, Eq. 83) plus a chunk-sized H psi scratch and grid fields.  Uses the current CUDA
 * device and the legacy default stream until lise_set_stream is called. */
int lise_create(int nx, int ny, int nz, double dx, double dt, int nwf_n, int nwf_p, lise_ctx **out);
/* lise_create with the line operator of the H-apply kernels chosen by the caller (for A/B checks of one kernel family
 * against another, or as a way out if one misbehaves on some driver): line_operator (HOST string) = "fft", "dmma",
 * "dense", or NULL / "auto" for lise_create's choice (see lise_line_operator below).  "dense" exists for every even
 * lattice; "fft" and "dmma" only for the lattices they were instantiated for, otherwise LISE_EUNSUPPORTED; an unknown
 * name is LISE_EINVAL.  All of them apply the same operator (Eqs. 48-50) and agree to round-off.  The automatic choice
 * falls back to "dense" by itself when the driver lacks cuTensorMapEncodeTiled, which the "fft" kernels need.
 * After a failed creation (either call) lise_last_error(NULL) returns the calling thread's message. */
int lise_create_with_line_operator(int nx, int ny, int nz, double dx, double dt, int nwf_n, int nwf_p,
                                   const char *line_operator, lise_ctx **out);
void lise_destroy(lise_ctx *ctx);

int lise_set_params(lise_ctx *ctx, const lise_params *p);
int lise_set_stream(lise_ctx *ctx, void *cuda_stream);       /* cudaStream_t owned by the caller */
/* Changes dt and restarts the multistep method (the next 3 steps use the starter). */
int lise_set_dt(lise_ctx *ctx, double dt);
/* Number of states processed per kernel launch (L2-resident batching of intermediates); <= 0 restores the default. */
int lise_set_chunk(lise_ctx *ctx, int nstates);
/* Tensor-core kernels only: enable (default) or disable running the
 * HBM-bound ABM update kernels on an internal second stream concurrently with the DMMA-bound kernels of the
 * neighbouring chunks.  Results are bit-identical either way.  All work is ordered back into the context's
 * stream before lise_step returns. */
int lise_set_overlap(lise_ctx *ctx, int enable);
/* Tensor-core kernels only: the densities of the new states are accumulated once per group of `nchunks` chunks
 * (default 8; <= 0 restores it): one density launch pair per group instead of one per chunk.  A scheduling choice;
 * results differ only by the summation order of the partial densities (round-off). */
int lise_set_density_group(lise_ctx *ctx, int nchunks);

/* Copies nwf_q states in (device pointer, layout above), accumulates their densities and resets the
 * multistep history, step counter and time. */
int lise_set_wavefunctions(lise_ctx *ctx, int species, const void *psi_dev);
int lise_get_wavefunctions(lise_ctx *ctx, int species, void *psi_dev);

/* HOST-buffer variants (psi_host is a HOST pointer, pinned or pageable, same layout): the copy is
 * enqueued on the context's stream with cudaMemcpyAsync.  lise_upload_wavefunctions with
 * keep_history = 0 is lise_set_wavefunctions from host memory; with keep_history = 1 it overwrites
 * y_n only (restoring a host mirror of the current wavefunctions, e.g. after a checkpoint,
 * PAPER.md:L764-L768), re-accumulates their densities and keeps the multistep history, step counter
 * and time.  lise_download_wavefunctions copies y_n out and returns after the stream has drained. */
int lise_upload_wavefunctions(lise_ctx *ctx, int species, const void *psi_host, int keep_history);
int lise_download_wavefunctions(lise_ctx *ctx, int species, void *psi_host);

/* Local densities of the current wavefunctions of one species in the layout of the paper's
 * d_densities (Table 2): 14*Nxyz doubles = n, tau, s(3), div J, j(3), curl j(3),
 * kappa (re, im).  Eq. 3 with tau via Eq. 51. */
int lise_densities(lise_ctx *ctx, int species, double *out14_dev);
/* Mean-field and pairing potentials of one species from the current densities of both species,
 * rows 0..13 of the paper's d_potentials (Table 3): U, hbar^2/2m*, lap(hbar^2/2m*),
 * W(3), S(3), A(3), Delta (re, im).  Eqs. 13-21 in the adopted reading. */
int lise_potentials(lise_ctx *ctx, int species, double *out14_dev);

/* out = H * in for nstates states of `species` (Eq. 11 with mu = 0; h of Eq. 12 in the lattice form
 * of Eqs. 55, 56), H built from the densities of the context's current wavefunctions of both
 * species.  No eta subtraction, no 1/(i hbar).  in_dev and out_dev must not overlap.  nstates = 0 is a
 * no-op (the pointers may then be null). */
int lise_apply_h(lise_ctx *ctx, int species, const void *in_dev, void *out_dev, int nstates);

/* Advances all states by nsteps time steps: the first 3 steps after lise_set_wavefunctions /
 * lise_set_dt use the 4th-order series expansion with predictor-corrector densities (Eqs. 75-77),
 * later steps the ABM predictor-modifier-corrector (Eq. 78 a-d) with 2 H evaluations per step and
 * the phase removal of Eqs. 80-81. */
int lise_step(lise_ctx *ctx, int nsteps);

/* State-sharded multi-GPU runs (one process per GPU: each rank owns nwf/G states,
 * grid fields replicated): the hook is called on the host at each of the two density barriers of a
 * step, after this rank's partial accumulators have been summed into `acc_dev` (DEVICE pointer,
 * `count` doubles = 2 species x 13 accumulators x Nxyz, work already enqueued on the context's
 * stream).  It must enqueue an in-place sum over ranks of acc_dev on the same stream (e.g. an NCCL
 * all-reduce) and return 0; a non-zero return aborts the step with LISE_ECUDA.  NULL removes the hook. */
typedef int (*lise_reduce_fn)(void *user, double *acc_dev, long count);
int lise_set_reduce_hook(lise_ctx *ctx, lise_reduce_fn fn, void *user);

/* Energy, particle numbers, norm / orthonormality defects of the current wavefunctions. Synchronises. */
int lise_observables(lise_ctx *ctx, lise_observables_t *host_out);
/* Eqs. 37-41 as grid reductions of the Table-2 / Table-3 fields of the current wavefunctions.  Synchronises. */
int lise_observables_ext(lise_ctx *ctx, lise_observables_ext_t *host_out);

/* Checkpoint / restart: a checkpoint is lise_download_wavefunctions (only the latest wavefunctions
 * are saved) plus the clock; a restart is lise_create + lise_upload_wavefunctions (keep_history = 0: the next three
 * steps go through the series expansion) + lise_set_time, which sets the clock (fm/c) and the step counter that
 * lise_observables reports, without touching the multistep start-up state. */
int lise_set_time(lise_ctx *ctx, double time, long step);

/* Boost (Eq. 23): u -> e^{i chi} u, v -> e^{-i chi} v for every state of the species; chi_dev: Nxyz doubles (DEVICE).
 * Re-accumulates the densities and restarts the multistep method (the next three steps use the starter). */
int lise_boost(lise_ctx *ctx, int species, const double *chi_dev);
/* External fields (Eq. 24): h_q -> h_q + U0 - (1/2) [Uvec . p + p . Uvec].  u0_dev: Nxyz doubles (MeV), uvec_dev:
 * 3 Nxyz doubles, component-major, in units of c; DEVICE pointers, copied into the context; NULL removes the field.
 * The copy made here is a spatial PROFILE; its time dependence (U(r,t), Uvec(r,t)) is the amplitude pair below.
 * Replacing the profile between steps instead would freeze the field during each step: first order in dt only. */
int lise_set_external_fields(lise_ctx *ctx, int species, const double *u0_dev, const double *uvec_dev);
/* Time-dependent external fields: U0(r, t) = f(t) U0(r), Uvec(r, t) = f(t) Uvec(r) for both species, with f_now = f(t_n) and
 * f_next = f(t_n + dt) supplied by the caller.  f_now multiplies the profiles wherever H is built from the current
 * wavefunctions y_n (first evaluation of Eq. 78, Eq. 75, lise_potentials, lise_apply_h, e_ext); f_next in the evaluation on the
 * modifier, which approximates y(t_{n+1}) (Eq. 78c); the start-up steps' corrector Hamiltonian, built from averaged
 * densities (Eq. 76), takes (f_now + f_next) / 2 (reading B33).  Default 1, 1 = a static field.  The pair holds
 * until it is set again, so a driven run calls this before every lise_step(ctx, 1); the frame terms are not scaled.
 * The ABM steps then keep their order (the oracle pin shows >= 4th order on a driven free state).  Non-finite: LISE_EINVAL. */
int lise_set_external_amplitudes(lise_ctx *ctx, double f_now, double f_next);
/* Moving and rotating frame (Eqs. 26, 36): h -> h - v_cm . p - omega . (l + s) for both species, l = (r - origin) x p;
 * v_cm_host in units of c, omega_host in c / fm, origin_host in fm (HOST pointers to 3 doubles; NULL = zero). */
int lise_set_frame(lise_ctx *ctx, const double *v_cm_host, const double *omega_host, const double *origin_host);
/* lise_potentials returns the fields that enter H: U includes U0, A includes -(hbar c / 2) (Uvec + v_cm + omega x r),
 * S includes -(hbar c / 2) omega. */

/* Per-kernel-class device timing with CUDA events on the context's stream (for bench.py's roofline).
 * lise_profile(ctx, 1) starts recording an event pair around every launch of the per-state kernels
 * (and around each grid-only phase); lise_profile_read synchronises and returns the summed
 * milliseconds and launch counts per class, then clears the record.  Classes:
 *   0 H-apply on yz-planes (y and z lines), 1 H-apply on xz-planes (x lines, eta),
 *   2 ABM update (generic kernels: + y/z density pass), 3 x density pass, 4 grid-only phase (reduction,
 *   potentials, Coulomb), 5 pointwise + y/z density pass (tensor-core kernels only).
 * Each pair is recorded on the stream its kernel is launched on (the update kernels run on an internal second
 * stream when overlap is on, see lise_set_overlap), so class times may overlap in wall time.
 * ms and counts are HOST arrays of 6 entries. */
int lise_profile(lise_ctx *ctx, int enable);
int lise_profile_read(lise_ctx *ctx, double *ms, long *counts);

/* Measures the fp64 FMA throughput of the current device (the denominator of the "alu" roofline): runs a
 * register-only DFMA kernel back to back on `stream` (cudaStream_t, may be NULL) for about `seconds`
 * and writes the best TFLOP/s (2 flop per FMA) seen in the second half of that time to *tflops_host
 * (HOST pointer).  sm_mhz_host is reserved (set to 0).  Synchronises. */
int lise_measure_fp64_peak(void *stream, double seconds, double *tflops_host, double *sm_mhz_host);

/* Which line operator the H-apply kernels of this context use: "fft" (one real line per thread, generated
 * real-input FFT code, Eqs. 49-50; lattices with every edge in {8, 12, 16, 20, 24, 32}), "dmma" (block-diagonalised
 * circulant on fp64 tensor-core tiles; the other lattice shapes the library was instantiated for) or "dense" (generic
 * DFMA circulant sums, any even lattice).  All three apply the same operator (Eqs. 48-50). */
const char *lise_line_operator(const lise_ctx *ctx);
/* Host-only: the number of fp64 instructions (DADD + DMUL + DFMA) of the generated straight-line FFT code for one
 * REAL line of n points: inner = (a = D x, b = D2 x), outer = (c = D g + D2 q); both 0 if no code was generated for n.
 * bench.py uses them for its model of the executed (as opposed to algorithmic) fp64 work. */
int lise_line_operator_cost(int n, int *inner_ops_host, int *outer_ops_host);

/* Host-only (no CUDA call, works without a GPU): the block-diagonalised form of the lattice derivative matrices
 * D (Eq. 48a) and D2 (Eq. 48b, prefactor as DESIGN.md B3) of a periodic line of n points (n % 4 == 0) that the
 * tensor-core kernels use.  dims_host (HOST, 5 ints) receives H (block size), R = n / H, J = R / 2 + 1 (blocks),
 * ND (entries per Toeplitz table) and the table length; tab_host (HOST, may be NULL to query the sizes, else at
 * least dims[4] doubles as stated by cap) receives tab[((op * J + j) * 2 + pq) * ND + d + H - 1] with op = 0 (D),
 * 1 (D2), pq = 0 (P_j), 1 (Q_j), d = r - r' in (-H, H):
 *   P_j[d] = (w_j / R) sum_p cos(2 pi j p / R) c[(d + H p) mod n],  Q_j with sin,  w_j = 1 for j = 0, R/2, else 2,
 * so that with b_j = sum_m cos(2 pi j m / R) x[r' + H m], e_j likewise with sin, S_j = P_j b_j - Q_j e_j,
 * T_j = P_j e_j + Q_j b_j:  (C x)[r + H m] = sum_j cos(2 pi j m / R) S_j[r] + sin(2 pi j m / R) T_j[r]. */
int lise_line_operator_tables(int n, double dx, double *tab_host, int cap, int *dims_host);

/* Renormalisation without a context and without any allocation ("normalise every qpwf" against the
 * slow loss of norm to round-off; the same operation lise_params.renormalize applies inside lise_step).
 *
 *   psi_k <- psi_k / sqrt(dV * sum_i |psi_k[i]|^2)      for k = 0 .. nstates-1, in place.
 *
 * For whom: code that holds the wavefunctions itself and cannot let a library allocate -- a run sized to fill the GPU
 * (wavefunctions + multistep history take nearly all of HBM, typically out of the application's own memory pool, so a
 * late cudaMalloc fails), or a time loop that cannot afford the device-wide stall of cudaMalloc / cudaFree.  Every
 * other call here needs a context, and lise_create allocates.  This call performs no cudaMalloc, no cudaFree and calls
 * no library routine that allocates; its per-state scratch (one double per state) is a fixed array inside liblise.so.
 *
 * Arguments: psi_dev DEVICE pointer, caller-owned, nstates * state_len interleaved complex128, state k at offset
 *   k * state_len (for the block layout above state_len = 4 * nx * ny * nz); dV > 0 the volume element; cuda_stream a
 *   cudaStream_t owned by the caller (NULL = legacy default stream).  The call only enqueues two kernels on that stream
 *   and returns; it does not synchronise.  A state that is identically zero is left unchanged.  nstates = 0 is a no-op.
 * Limit: nstates <= LISE_STATIC_MAX_STATES.  More is refused with LISE_EINVAL (nothing is enqueued) and
 *   lise_static_last_error() says so; renormalise a longer array slice by slice.
 * Cost: the array (LISE_STATIC_MAX_STATES doubles, 128 KB) occupies device memory on every GPU on which this library's
 *   CUDA code is loaded, for the life of the process, used or not.
 * First call on a device: it looks up the array's address on the current device (cudaGetSymbolAddress, which may have
 *   to load the library's CUDA module there) and caches it; later calls on that device skip this.  Make that first call
 *   during set-up, with the intended device current and before any stream capture is begun on the thread.
 * Sharing: there is ONE array per device for all callers.  Each call overwrites entries 0 .. nstates-1 before it reads
 *   them, so nothing has to be cleared between calls and whatever an earlier call left behind is never read.  Calls
 *   enqueued on the same stream run one after the other and are safe.  Two calls that can run at the same time on one
 *   device (different streams without an event between them, two host threads on different streams) race on the array
 *   and give wrong norms: order them yourself.
 * Errors: LISE_EINVAL (null psi_dev, negative nstates, state_len <= 0, dV not positive and finite, nstates over the
 *   limit), LISE_ECUDA (address lookup or launch failed), LISE_EUNSUPPORTED (device ordinal >= 64).  The message of the
 *   calling thread's last failure is lise_static_last_error() (HOST string owned by the library, "" after a success). */
#define LISE_STATIC_MAX_STATES 16384
int lise_renormalize_static(void *psi_dev, int nstates, long long state_len, double dV, void *cuda_stream);
const char *lise_static_last_error(void);

/* Number of kernel launches issued by this context so far (for bench.py's gpu_launches). */
long lise_launch_count(const lise_ctx *ctx);
/* Bytes of device memory held by the context. */
long long lise_device_bytes(const lise_ctx *ctx);

const char *lise_strerror(int code);
const char *lise_last_error(const lise_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
