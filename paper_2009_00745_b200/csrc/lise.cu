// lise.cu -- C-ABI entry points (include/lise.h) and host-side orchestration of the TDSLDA step.
//
// Resident state arrays per species ("slots", roles rotate by pointer swap):
//   A y_n | B y_{n-1} -> Q -> y_{n+1} | C f_{n-3} -> f_n | D f_{n-1} | E f_{n-2} | F e_n -> e_{n+1} | G m
// One ABM step (Eq. 78) = two evaluations; each evaluation = grid-only potentials, then per
// chunk of states: k_happly<0> (yz-planes) -> k_happly<1> (xz-planes, eta) -> k_update_yz (ABM + y/z
// densities of the new state) -> k_dens_x (x densities of the new state).
#include "common.cuh"
#include "state_kernels.cuh"
#include "plane5_kernels.cuh"
#include "fft_plane_kernels.cuh"
#include "grid_kernels.cuh"
#include "peak_kernels.cuh"
#include <mutex>
#include <new>
#include <stdlib.h>
#include <vector>

enum { RA = 0, RB, RC, RD, RE, RF, RG };

typedef void (*HKern)(HArgs);
typedef void (*UKern)(UArgs);
typedef void (*DKern)(DArgs);
struct KernSet {
    HKern h_yz, h_xz;
    UKern u[4];
    DKern d_x, d_yz;                       // d_yz: plane5 kernels only (the generic update kernel carries the y/z densities)
    const char* name;
    int v5;                                // plane5 kernel set: pure-streaming update + separate density kernels
    int thr_h[2], thr_u, thr_d, thr_dyz;   // threads per CTA: happly yz / xz, update, dens_x, dens_yz
    size_t smem_h[2], smem_u, smem_d, smem_dyz;   // dynamic shared memory, bytes (0 = filled by ctx_init for the generic path)
    int ups_xz;                            // eta partial sums per state = ups_xz * ny
    int cps_h[2];                          // resident CTAs per SM of the two H-apply kernels (state groups = G * cps)
    int tma_h[2];                          // the H-apply kernel stages its planes by tensor-map copies (needs HArgs::tmX)
};
struct lise_ctx {
    Lattice L;
    int n[3];
    double dt;
    int nwf[2];
    lise_params par;
    PhysConst pc;
    cudaStream_t stream;
    double2* ctab[3];
    double* stab[3];                        // block-diagonalised line-operator tables (split_lineop.cuh)
    cudaStream_t stream2;                   // the HBM-bound update kernels run here (lowest priority), overlapping the DMMA kernels
    cudaStream_t streamH;                   // highest priority: the DMMA kernels of lise_step run here when overlap is on, so
                                            // that their CTAs are placed first and the update CTAs fill the room left beside them
    cudaEvent_t ev_fork, ev_join;
    cudaStream_t user_stream; int user_stream_valid;   // the caller's stream while lise_step runs on streamH
    cudaEvent_t ev_h[2], ev_u[2];
    int overlap, dgroup;                    // dgroup: chunks per density-kernel launch
    cplx* slot[2][LISE_NSLOT];
    int role[LISE_NSLOT];
    cplx* W;                                // [2][wcap] states: H-apply output, double-buffered across chunks
    int chunk, wcap;
    double *eta_part, *eta_fix;             // eta_part: [2][wcap][neta]
    int G;
    double *part[2], *acc[2], *acc0[2], *dens[2], *pot[2], *geff[2];
    double *gtmp, *phi;
    GJob *jobs1, *jobs2;
    int njobs1, njobs2;
    int P; double Dc;
    cplx *tw, *cA1, *cA2, *cA3;
    double* ebuf; int eblocks;
    cplx* ovl;
    int R, mma;
    double amp_now, amp_next;               // amplitudes of the Eq. 24 fields at t_n and t_{n+1} (lise_set_external_amplitudes)
    int lop_mode;                           // LOP_* requested at creation (lise_create_with_line_operator)
    KernSet ks;
    int have[2], pot_valid;
    long step; double time;
    long since;                             // steps since the multistep method was (re)started: < 3 -> starter
    double *uext[2], *vext[2];              // external fields of Eq. 24 in use (NULL = none) ...
    double *uext_buf[2], *vext_buf[2];      // ... and the context's buffers that hold them
    double* mbuf; double* nrm;              // reduction scratch of the Eq. 37-41 observables; state norms (renormalisation)
    long launches; long long bytes;
    std::vector<void*>* allocs;
    // optional per-kernel-class timing with CUDA events on the context's stream (lise_profile)
    lise_reduce_fn reduce_fn; void* reduce_user;
    int prof; int prof_n;
    std::vector<cudaEvent_t>* prof_ev;      // pairs (start, stop)
    std::vector<int>* prof_cls;
    char err[256];
};

enum { PC_HAPPLY_YZ = 0, PC_HAPPLY_XZ, PC_UPDATE, PC_DENS_X, PC_GRID, PC_DENS_YZ, PC_NCLASS };

static void prof_begin(lise_ctx* c, int cls, cudaStream_t st = nullptr)
{
    if (!c->prof) return;
    if (!st) st = c->stream;
    if ((size_t)(2 * c->prof_n + 2) > c->prof_ev->size()) {
        cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
        c->prof_ev->push_back(a); c->prof_ev->push_back(b); c->prof_cls->push_back(cls);
    }
    (*c->prof_cls)[c->prof_n] = cls;
    cudaEventRecord((*c->prof_ev)[2 * c->prof_n], st);
}
static void prof_end(lise_ctx* c, cudaStream_t st = nullptr)
{
    if (!c->prof) return;
    if (!st) st = c->stream;
    cudaEventRecord((*c->prof_ev)[2 * c->prof_n + 1], st);
    c->prof_n++;
}

static const char* g_noctx = "no context";

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            snprintf(c->err, sizeof(c->err), "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return (e_ == cudaErrorMemoryAllocation) ? LISE_ENOMEM : LISE_ECUDA;                   \
        }                                                                                          \
    } while (0)
#define CKL()                                                                                      \
    do { c->launches++; CK(cudaGetLastError()); } while (0)
#define TRY(expr) do { int rc_ = (expr); if (rc_ != LISE_OK) return rc_; } while (0)

// nothing may throw across the C ABI: host allocations (std::vector, new) inside an entry point run under this guard
template <class F>
static int guarded(F&& f)
{
    try { return f(); }
    catch (const std::bad_alloc&) { return LISE_ENOMEM; }
    catch (...) { return LISE_ECUDA; }
}

static int dmalloc(lise_ctx* c, void** p, size_t bytes)
{
    if (bytes == 0) bytes = 16;
    CK(cudaMalloc(p, bytes));
    c->allocs->push_back(*p);
    c->bytes += (long long)bytes;
    return LISE_OK;
}
#define DM(ptr, count) TRY(dmalloc(c, (void**)&(ptr), sizeof(*(ptr)) * (size_t)(count)))

static inline unsigned nblk(size_t n, int t) { return (unsigned)((n + t - 1) / t); }
static inline cplx* S(lise_ctx* c, int q, int r) { return c->slot[q][c->role[r]]; }

// ---- tables: closed-form DVR coefficients (Eq. 48a; Eq. 48b with prefactor 2 pi^2 / (N a)^2) ----
static void host_ctab(int N, double a, std::vector<double2>& t)
{
    std::vector<double> c1(N), c2(N);
    const long double pi = 3.14159265358979323846264338327950288L;
    c1[0] = 0.0;
    c2[0] = (double)(-pi * pi / (3.0L * a * a) * (1.0L + 2.0L / ((long double)N * N)));
    for (int k = 1; k < N; ++k) {
        long double th = pi * k / N;
        long double sgn = (k % 2) ? -1.0L : 1.0L;
        c1[k] = (2 * k == N) ? 0.0 : (double)(pi / (N * (long double)a) * sgn * cosl(th) / sinl(th));
        c2[k] = (double)(-2.0L * pi * pi / ((long double)N * N * a * a) * sgn / (sinl(th) * sinl(th)));
    }
    t.resize(2 * N);
    for (int d = -N; d < N; ++d) {
        int k = ((d % N) + N) % N;
        t[N + d] = make_double2(c1[k], c2[k]);
    }
}

// ---- block-diagonalised tables of split_lineop.cuh: tab[((op * J + j) * 2 + pq) * ND + d + H - 1] ----
struct LOpDims { int N, H, R, J, NTH, NKH, ND, TABSZ; };
static LOpDims lop_dims(int N)
{
    LOpDims d;
    d.N = N; d.H = (N % 8 == 0 && N >= 16 && N / 8 <= LISE_RMAX) ? 8 : N;
    d.R = N / d.H; d.J = d.R / 2 + 1; d.NTH = (d.H + 7) / 8; d.NKH = d.H / 4;
    d.ND = d.H + 8 * d.NTH - 1; d.TABSZ = 2 * d.J * 2 * d.ND;
    return d;
}
static void host_stab(int N, double a, std::vector<double>& tab)
{
    std::vector<double2> ct;
    host_ctab(N, a, ct);                       // ct[N + d] = (c1, c2)[d mod N]
    const LOpDims D = lop_dims(N);
    const long double pi = 3.14159265358979323846264338327950288L;
    tab.assign(D.TABSZ, 0.0);
    for (int op = 0; op < 2; ++op)
        for (int j = 0; j < D.J; ++j) {
            const long double w = (j == 0 || 2 * j == D.R) ? 1.0L : 2.0L;
            for (int d = -(D.H - 1); d < D.H; ++d) {           // d >= H: padding rows, left 0
                long double P = 0.0L, Q = 0.0L;
                for (int p = 0; p < D.R; ++p) {
                    const int k = (((d + D.H * p) % N) + N) % N;
                    const long double cv = op ? ct[N + k].y : ct[N + k].x;
                    const int jp = (j * p) % D.R;
                    const long double th = 2.0L * pi * jp / D.R;
                    const long double co = (4 * jp == D.R || 4 * jp == 3 * D.R) ? 0.0L : cosl(th);
                    const long double si = (jp == 0 || 2 * jp == D.R) ? 0.0L : sinl(th);
                    P += co * cv; Q += si * cv;
                }
                tab[((op * D.J + j) * 2 + 0) * D.ND + d + D.H - 1] = (double)(w / D.R * P);
                tab[((op * D.J + j) * 2 + 1) * D.ND + d + D.H - 1] = (double)(w / D.R * Q);
            }
        }
}
// generic real-DFT coefficients in constant memory: c_rdft[R][q][m] (spectral order of split_lineop.cuh)
static int upload_rdft()
{
    static double h[LISE_RMAX + 1][LISE_RMAX][LISE_RMAX];
    const long double pi = 3.14159265358979323846264338327950288L;
    memset(h, 0, sizeof(h));
    for (int R = 1; R <= LISE_RMAX; ++R)
        for (int q = 0; q < R; ++q) {
            int j; bool sn;
            if (q == 0) { j = 0; sn = false; }
            else if (R % 2 == 0 && q == R - 1) { j = R / 2; sn = false; }
            else { j = (q + 1) / 2; sn = (q % 2 == 0); }
            for (int m = 0; m < R; ++m) {
                const int jm = (j * m) % R;
                const long double th = 2.0L * pi * jm / R;
                long double v;
                if (sn) v = (jm == 0 || 2 * jm == R) ? 0.0L : sinl(th);
                else    v = (4 * jm == R || 4 * jm == 3 * R) ? 0.0L : cosl(th);
                h[R][q][m] = (double)v;
            }
        }
    return cudaMemcpyToSymbol(c_rdft, h, sizeof(h)) == cudaSuccess ? LISE_OK : LISE_ECUDA;
}

static void set_physconst(lise_ctx* c)
{
    const lise_params& p = c->par;
    PhysConst& k = c->pc;
    k.h2m = p.hbar2_2m; k.e2 = p.e2; k.hbarc = p.hbarc; k.gamma = p.gamma; k.a = c->L.dx;
    k.Kc = 2.442749607806335;
    if (p.functional == 1) {
        // SeaLL1 (Eq. 10): volume term by its own coefficients, gradient and spin-orbit couplings supplied, m* = m
        for (int t = 0; t < 2; ++t) { k.Cn[t] = k.Cg[t] = k.Ct[t] = 0.0; k.Cd[t] = p.sea_cdn[t]; k.CJ[t] = p.sea_cdj[t]; }
    } else {
        // couplings of Eq. 9 from the Skyrme parameters (standard relations, DESIGN.md A.0)
        k.Cn[0] = 3.0 * p.t0 / 8.0;                       k.Cn[1] = -(p.t0 / 4.0) * (0.5 + p.x0);
        k.Cg[0] = p.t3 / 16.0;                            k.Cg[1] = -(p.t3 / 24.0) * (0.5 + p.x3);
        k.Cd[0] = -9.0 * p.t1 / 64.0 + (p.t2 / 16.0) * (1.25 + p.x2);
        k.Cd[1] = (3.0 * p.t1 / 32.0) * (0.5 + p.x1) + (p.t2 / 32.0) * (0.5 + p.x2);
        k.Ct[0] = 3.0 * p.t1 / 16.0 + (p.t2 / 4.0) * (1.25 + p.x2);
        k.Ct[1] = -(p.t1 / 8.0) * (0.5 + p.x1) + (p.t2 / 8.0) * (0.5 + p.x2);
        k.CJ[0] = -3.0 * p.W0 / 4.0;                      k.CJ[1] = -p.W0 / 4.0;
    }
    k.g0[0] = p.g0_n; k.g0[1] = p.g0_p;
    k.alpha = p.alpha_pair; k.mu[0] = p.mu_n; k.mu[1] = p.mu_p; k.ecut = p.e_cut;
    for (int j = 0; j < 3; ++j) { k.sa[j] = p.sea_a[j]; k.sb[j] = p.sea_b[j]; k.sc[j] = p.sea_c[j]; }
    k.coulomb = p.coulomb; k.rearr = p.pairing_rearrangement; k.functional = p.functional; k.cutoff = p.pairing_cutoff;
}

extern "C" int lise_default_params(lise_params* p)
{
    if (!p) return LISE_EINVAL;
    p->hbar2_2m = 20.73553; p->e2 = 1.439964; p->hbarc = 197.3269804;
    p->t0 = -2488.91; p->t1 = 486.82; p->t2 = -546.39; p->t3 = 13777.0;
    p->x0 = 0.834; p->x1 = -0.344; p->x2 = -1.000; p->x3 = 1.354;
    p->gamma = 1.0 / 6.0; p->W0 = 123.0;
    p->g0_n = -250.0; p->g0_p = -250.0;
    p->coulomb = 1; p->pairing_rearrangement = 1; p->remove_phase = 1;
    p->alpha_pair = 0.0; p->mu_n = p->mu_p = 0.0; p->e_cut = 0.0;
    for (int j = 0; j < 3; ++j) p->sea_a[j] = p->sea_b[j] = p->sea_c[j] = 0.0;
    p->sea_cdn[0] = p->sea_cdn[1] = p->sea_cdj[0] = p->sea_cdj[1] = 0.0;
    p->functional = 0; p->pairing_cutoff = 0; p->renormalize = 0;
    return LISE_OK;
}

// ---- kernel sets: the plane kernels instantiated for one line-operator policy per plane kind ----
template <class LOYZ, class LOXZ>
static KernSet make_set(const char* name)
{
    KernSet k;
    k.h_yz = k_happly<0, LOYZ>; k.h_xz = k_happly<1, LOXZ>;
    k.u[0] = k_update_yz<0, LOYZ>; k.u[1] = k_update_yz<1, LOYZ>; k.u[2] = k_update_yz<2, LOYZ>; k.u[3] = k_update_yz<3, LOYZ>;
    k.d_x = k_dens_x<LOXZ>; k.d_yz = nullptr;
    k.name = name; k.v5 = 0;
    return k;
}
// ---- plane5 kernels: compile-time choice of unit size (NCOMP), prefetch depth (NBUF), warps, staging ----
static constexpr size_t SMEM_LIMIT = 227 * 1024;
template <int N> static constexpr size_t tabsz() { return (size_t)LOp<N>::TABSZ; }
template <int NY, int NZ>
static constexpr size_t v5_smem_happly_yz(int ncomp, int nbuf, bool vstage)
{
    return 8 * ((tabsz<NY>() + tabsz<NZ>() + 1) / 2 * 2) + 16 * (size_t)(NY * ldpad(NZ)) * ncomp * (nbuf + 1)
         + 8 * (size_t)(NY * ldpad(NZ)) * (6 + (vstage ? 6 : 0));
}
template <int NX, int NZ>
static constexpr size_t v5_smem_happly_xz(int ncomp, int nbuf, int nwarp, bool wst = false)
{
    return 8 * ((tabsz<NX>() + 1) / 2 * 2) + 16 * (size_t)(NX * ldpad(NZ)) * ncomp * nbuf * (wst ? 2 : 1) + 8 * (size_t)(NX * ldpad(NZ)) * 4 + 8 * 2 * nwarp;
}
template <int NY, int NZ>
static constexpr size_t v5_smem_dens_yz(int sb) { return 8 * ((tabsz<NY>() + tabsz<NZ>() + 1) / 2 * 2) + 16 * (size_t)(4 * sb * NY * ldpad(NZ)); }
template <int NX, int NZ>
static constexpr size_t v5_smem_dens_x(int sb) { return 8 * ((tabsz<NX>() + 1) / 2 * 2) + 16 * (size_t)(4 * sb * NX * ldpad(NZ)); }
// states per barrier round of a density kernel: up to 4, as many as fit half of the shared memory 
template <int N1, int NZ>
static constexpr int v5_dens_sb() { return (16 * (size_t)(4 * 4 * N1 * ldpad(NZ)) <= 180 * 1024) ? 4 : (16 * (size_t)(4 * 2 * N1 * ldpad(NZ)) <= 180 * 1024) ? 2 : 1; }
static constexpr int imin(int a, int b) { return a < b ? a : b; }
static constexpr int imax(int a, int b) { return a > b ? a : b; }
// warps per 2-spinor of an H-apply CTA: one strip task per warp if possible; long lines need more registers per thread
// warps a CTA may have for lines of `nline` points (long lines need more registers per thread)
static constexpr int v5_wcap(int nline) { return nline >= 48 ? 8 : nline >= 40 ? 10 : 12; }
static constexpr int v5_wpp(int npair, int strips, int nline) { return imin(strips, v5_wcap(nline) / npair); }

static constexpr int v6_regs(int warps) { return fft_full_regs(warps); }
// register cap of a DMMA H-apply kernel with `warps` warps and `ctas` CTAs per SM: what leaves room for the co-resident
// update CTA (plane_common.cuh: coresident_regs, the budget is per SM sub-partition)
static constexpr int v5_maxr(int warps, int ctas) { return coresident_regs(warps * ctas); }
// warps for `tasks` equal tasks per pass: all of them if they fit under `cap`, else the largest count <= cap that
// divides them evenly
static constexpr int v5_warps(int tasks, int cap)
{
    if (tasks <= cap) return tasks;
    for (int w = cap; w >= cap / 2; --w) if (tasks % w == 0) return w;
    return cap;
}
// one plane-owner CTA per SM, whole states per unit if shared memory allows.  HAPPLY = false: only the update and density
// kernels (the FFT kernel sets bring their own H-apply kernels).
template <int NX, int NY, int NZ, bool HAPPLY = true>
static KernSet make_v5_set()
{
    KernSet k;
    k.h_yz = nullptr; k.h_xz = nullptr;
    k.cps_h[0] = k.cps_h[1] = 1; k.tma_h[0] = k.tma_h[1] = 0;
    k.thr_h[0] = k.thr_h[1] = 0; k.smem_h[0] = k.smem_h[1] = 0; k.ups_xz = 1;
    if constexpr (HAPPLY) {
        // yz: prefer whole states with prefetch, then 2-spinors with prefetch, then 2-spinors without
        constexpr int CYZ = (v5_smem_happly_yz<NY, NZ>(4, 2, false) <= SMEM_LIMIT) ? 4 : 2;
        constexpr int BYZ = (v5_smem_happly_yz<NY, NZ>(CYZ, 2, false) <= SMEM_LIMIT) ? 2 : 1;
        constexpr bool VST = v5_smem_happly_yz<NY, NZ>(CYZ, BYZ, true) <= SMEM_LIMIT;
        constexpr int WYZ = (CYZ / 2) * v5_wpp(CYZ / 2, imax(NY, NZ) / 4, imax(NY, NZ));
        constexpr int WXZ0 = 12;
        constexpr int CXZ = (v5_smem_happly_xz<NX, NZ>(4, 2, WXZ0) <= SMEM_LIMIT) ? 4 : 2;
        constexpr int BXZ = (v5_smem_happly_xz<NX, NZ>(CXZ, 2, WXZ0) <= SMEM_LIMIT) ? 2 : 1;
        constexpr int WXZ = v5_warps((CXZ / 2) * NZ / 4, NX == 32 ? 8 : v5_wcap(NX));
        static_assert(v5_smem_happly_yz<NY, NZ>(CYZ, BYZ, VST) <= SMEM_LIMIT, "yz plane too large");
        static_assert(v5_smem_happly_xz<NX, NZ>(CXZ, BXZ, WXZ) <= SMEM_LIMIT, "xz plane too large");
        // register caps: the co-resident budget (room for the update CTA); a yz kernel of 10 or more warps takes the whole
        // register file instead (at 144 registers its spills cost more than the overlap gains: 40^3, measured)
        constexpr int RYZ = WYZ >= 10 ? v6_regs(WYZ) : v5_maxr(WYZ, 1), RXZ = v5_maxr(WXZ, 1);
        constexpr bool WST = BXZ == 2 && v5_smem_happly_xz<NX, NZ>(CXZ, BXZ, WXZ, true) <= SMEM_LIMIT;
        k.h_yz = k5_happly_yz<NY, NZ, CYZ, BYZ, WYZ, VST, RYZ>; k.h_xz = k5_happly_xz<NX, NZ, CXZ, BXZ, WXZ, RXZ, WST>;
        k.thr_h[0] = 32 * WYZ; k.thr_h[1] = 32 * WXZ;
        k.smem_h[0] = v5_smem_happly_yz<NY, NZ>(CYZ, BYZ, VST); k.smem_h[1] = v5_smem_happly_xz<NX, NZ>(CXZ, BXZ, WXZ, WST);
        k.ups_xz = 4 / CXZ;
    }
    constexpr int WDY = imin(2 * (NY / 4) + 2 * (NZ / 4), imax(NY, NZ) >= 40 ? 8 : 12);
    constexpr int WDX = imin(2 * NZ / 4, NX >= 40 ? 8 : 12);
    k.u[0] = nullptr; k.u[1] = k5_update<1>; k.u[2] = k5_update<2>; k.u[3] = k5_update<3>;
    constexpr int SBY = v5_dens_sb<NY, NZ>(), SBX = v5_dens_sb<NX, NZ>();
    k.d_yz = k5_dens_yz<NY, NZ, WDY, SBY>; k.d_x = k5_dens_x<NX, NZ, WDX, SBX>;
    k.name = "dmma"; k.v5 = 1;
    k.thr_u = LISE_UPD_THREADS; k.thr_d = 32 * WDX; k.thr_dyz = 32 * WDY;
    k.smem_u = 0; k.smem_d = v5_smem_dens_x<NX, NZ>(SBX); k.smem_dyz = v5_smem_dens_yz<NY, NZ>(SBY);
    return k;
}
// ---- FFT-cost line operator (fft_plane_kernels.cuh): one real line per thread, generated real-input FFT codelets.
// Lattices with every edge in {8, 12, 16, 20, 24, 32}.  Both H-apply kernels are the FFT ones; where a whole state fits
// the yz-plane CTA's shared memory (edges <= 24) the yz kernel adds the pairing block, else (32^3, 2-spinor units) the
// xz kernel does.  The ABM update and the density kernels are those of plane5_kernels.cuh.
template <int NX, int NY, int NZ>
static KernSet make_v6_set()
{
    KernSet k = make_v5_set<NX, NY, NZ, false>();              // update and density kernels
    constexpr int CYZ = (YZGeom<NY, NZ, 4>::SMEM <= SMEM_LIMIT) ? 4 : 2;
    typedef YZGeom<NY, NZ, CYZ> GY;
    typedef XZGeom<NX, NZ> GX;
    static_assert(GY::SMEM <= SMEM_LIMIT, "yz plane too large");
    static_assert(GX::SMEM <= SMEM_LIMIT, "xz plane too large");
    constexpr bool WHOLE = (CYZ == 4);                         // the yz kernel sees whole states: it adds the pairing block
    // the yz kernel takes every register of the SM (its shared-memory pipe is the busiest unit: nothing gains from a
    // neighbour); the xz kernel leaves one warp of LISE_UPD_REGS registers per sub-partition to the update CTA
    if constexpr (WHOLE) k.h_yz = k6_yz_whole<NY, NZ>();       // own translation unit (happly_yz_whole.cu)
    else k.h_yz = k6_happly_yz<NY, NZ, CYZ, v6_regs(GY::NW), false>;
    k.cps_h[0] = 1; k.thr_h[0] = 32 * GY::NW; k.smem_h[0] = GY::SMEM; k.tma_h[0] = 1;
    k.h_xz = k6_happly_xz<NX, NZ, coresident_regs(GX::NW), !WHOLE>;
    k.cps_h[1] = 1; k.thr_h[1] = 32 * GX::NW; k.smem_h[1] = GX::SMEM; k.ups_xz = 1; k.tma_h[1] = 1;
    k.name = "fft";
    return k;
}
#define LISE_FFT_SHAPES(X) \
    X(8, 8, 8) X(12, 12, 12) X(16, 16, 16) X(20, 20, 20) X(24, 24, 24) X(32, 32, 32) X(12, 8, 16) X(16, 12, 8) X(12, 12, 16)

// The DMMA H-apply kernels are instantiated for the lattices the FFT kernels do not cover: 40^3 (BASELINE.json config 4),
// the paper's 24^2 x 48 and 24^2 x 64 (config 3).  Anything else runs the generic DFMA kernels.
#define LISE_MMA_SHAPES(X) X(40, 40, 40) X(24, 24, 48) X(24, 24, 64)
// mode: LOP_AUTO picks the fastest set instantiated for the lattice; LOP_FFT / LOP_DMMA only that family (false and
// out->name = nullptr if the lattice has none); LOP_DENSE the generic kernels (lise_create_with_line_operator)
enum { LOP_AUTO = 0, LOP_FFT = 1, LOP_DMMA = 2, LOP_DENSE = 3 };
static bool pick_kernels(int nx, int ny, int nz, int R, KernSet* out, int mode = LOP_AUTO)
{
    if (mode == LOP_AUTO || mode == LOP_FFT) {
#define X(a, b, c_) if (nx == a && ny == b && nz == c_) { *out = make_v6_set<a, b, c_>(); return true; }
        LISE_FFT_SHAPES(X)
#undef X
    }
    if (mode == LOP_AUTO || mode == LOP_DMMA) {
#define X(a, b, c_) if (nx == a && ny == b && nz == c_) { *out = make_v5_set<a, b, c_>(); return true; }
        LISE_MMA_SHAPES(X)
#undef X
    }
    if (mode == LOP_FFT || mode == LOP_DMMA) { out->name = nullptr; return false; }
    if (R == 8) *out = make_set<DenseLines<8>, DenseLines<8>>("dense");
    else if (R == 4) *out = make_set<DenseLines<4>, DenseLines<4>>("dense");
    else *out = make_set<DenseLines<2>, DenseLines<2>>("dense");
    out->thr_h[0] = out->thr_h[1] = out->thr_u = out->thr_d = out->thr_dyz = 0;
    out->smem_h[0] = out->smem_h[1] = out->smem_u = out->smem_d = out->smem_dyz = 0;
    out->ups_xz = 1; out->v5 = 0; out->d_yz = nullptr; out->cps_h[0] = out->cps_h[1] = 1; out->tma_h[0] = out->tma_h[1] = 0;
    return false;
}

// tensor map of a wavefunction block X = [ncomp][nx][ny][nz] complex128 for the plane-tile loads of the FFT kernels:
// elements are doubles, innermost box = 16 doubles = one 128-byte swizzle row; KIND 0: [ny rows][128 B] tiles of a
// yz-plane, KIND 1: [nx rows][128 B] tiles of an xz-plane (rows at stride ny nz)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
// cuTensorMapEncodeTiled through the runtime's driver entry point query (no link against libcuda), resolved once per
// process under a lock; nullptr if this driver does not provide it (ctx_init then falls back to the generic kernels)
static EncodeTiledFn resolve_encode_tiled()
{
    static std::mutex mu;
    static int state = 0;                          // 0 not tried, 1 found, -1 missing
    static EncodeTiledFn encode = nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (state == 0) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres = cudaDriverEntryPointSymbolNotFound;
        const cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e == cudaSuccess && fn && qres == cudaDriverEntryPointSuccess) { encode = (EncodeTiledFn)fn; state = 1; }
        else { (void)cudaGetLastError(); state = -1; }
    }
    return encode;
}
static int make_plane_tmap(lise_ctx* c, int kind, const cplx* X, int ncomp, CUtensorMap* out)
{
    const EncodeTiledFn encode = resolve_encode_tiled();
    if (!encode) { snprintf(c->err, sizeof(c->err), "cuTensorMapEncodeTiled not available"); return LISE_ECUDA; }
    const Lattice& L = c->L;
    const cuuint64_t dims[4] = {(cuuint64_t)2 * L.nz, (cuuint64_t)L.ny, (cuuint64_t)L.nx, (cuuint64_t)(ncomp > 0 ? ncomp : 1)};
    const cuuint64_t strides[3] = {(cuuint64_t)16 * L.nz, (cuuint64_t)16 * L.nz * L.ny, (cuuint64_t)16 * L.nxyz};
    const cuuint32_t box[4] = {16u, kind == 0 ? (cuuint32_t)L.ny : 1u, kind == 0 ? 1u : (cuuint32_t)L.nx, 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)X, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { snprintf(c->err, sizeof(c->err), "cuTensorMapEncodeTiled failed (%d)", (int)r); return LISE_ECUDA; }
    return LISE_OK;
}

template <int KIND>
static int launch_happly(lise_ctx* c, const HArgs& a)
{
    HArgs b = a;
    if (c->ks.tma_h[KIND]) TRY(make_plane_tmap(c, KIND, a.X, 4 * a.ns, &b.tmX));
    b.G = c->G * c->ks.cps_h[KIND];
    dim3 grid(KIND == 0 ? c->L.nx : c->L.ny, b.G);
    prof_begin(c, KIND == 0 ? PC_HAPPLY_YZ : PC_HAPPLY_XZ);
    (KIND == 0 ? c->ks.h_yz : c->ks.h_xz)<<<grid, c->ks.thr_h[KIND], c->ks.smem_h[KIND], c->stream>>>(b);
    prof_end(c);
    CKL();
    return LISE_OK;
}
// MODE 1, 2: ABM (Eq. 78); 3: starter Taylor term; 0: densities of u.Z only (generic kernels).  `st`: launch stream
template <int MODE>
static int launch_update(lise_ctx* c, const UArgs& a, cudaStream_t st)
{
    prof_begin(c, PC_UPDATE, st);
    if (c->ks.v5) {
        const size_t slen = (size_t)4 * c->L.nxyz, per = (size_t)LISE_UPD_THREADS * UpdEpt<MODE>::V;
        dim3 grid((unsigned)((slen + per - 1) / per), a.ns);
        c->ks.u[MODE]<<<grid, LISE_UPD_THREADS, 0, st>>>(a);
    } else {
        dim3 grid(c->L.nx, c->G);
        c->ks.u[MODE]<<<grid, c->ks.thr_u, c->ks.smem_u, st>>>(a);
    }
    prof_end(c, st);
    CKL();
    return LISE_OK;
}
static int launch_dens_x(lise_ctx* c, const DArgs& a)
{
    dim3 grid(c->L.ny, c->G);
    prof_begin(c, PC_DENS_X);
    c->ks.d_x<<<grid, c->ks.thr_d, c->ks.smem_d, c->stream>>>(a);
    prof_end(c);
    CKL();
    return LISE_OK;
}
static int launch_dens_yz(lise_ctx* c, const DArgs& a)
{
    dim3 grid(c->L.nx, c->G);
    prof_begin(c, PC_DENS_YZ);
    c->ks.d_yz<<<grid, c->ks.thr_dyz, c->ks.smem_dyz, c->stream>>>(a);
    prof_end(c);
    CKL();
    return LISE_OK;
}
static int set_attrs(lise_ctx* c)
{
    CK(cudaFuncSetAttribute(c->ks.h_yz, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->ks.smem_h[0]));
    CK(cudaFuncSetAttribute(c->ks.h_xz, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->ks.smem_h[1]));
    if (!c->ks.v5)
        for (int m = 0; m < 4; ++m) CK(cudaFuncSetAttribute(c->ks.u[m], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->ks.smem_u));
    CK(cudaFuncSetAttribute(c->ks.d_x, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->ks.smem_d));
    if (c->ks.d_yz) CK(cudaFuncSetAttribute(c->ks.d_yz, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->ks.smem_dyz));
    return LISE_OK;
}

static void fill_common(lise_ctx* c, const double2** ct) { for (int i = 0; i < 3; ++i) ct[i] = c->ctab[i]; }
static void fill_stab(lise_ctx* c, const double** st) { for (int i = 0; i < 3; ++i) st[i] = c->stab[i]; }
static inline int neta(const lise_ctx* c) { return c->ks.ups_xz * c->L.ny; }
static inline cplx* Wbuf(lise_ctx* c, int b) { return c->W + (size_t)b * c->wcap * 4 * c->L.nxyz; }
static inline double* etabuf(lise_ctx* c, int b) { return c->eta_part + (size_t)b * c->wcap * neta(c); }

// W = H X for ns states (ns <= chunk) of species q; eta partial sums -> eta (buffer of ns * neta doubles)
static int apply_h_chunk(lise_ctx* c, int q, const cplx* X, cplx* W, double* eta, int ns)
{
    HArgs a;
    a.L = c->L; a.X = X; a.W = W; a.pot = c->pot[q]; fill_common(c, a.ctab); fill_stab(c, a.stab);
    a.eta_part = eta; a.ns = ns; a.G = c->G;
    TRY(launch_happly<0>(c, a));
    TRY(launch_happly<1>(c, a));
    return LISE_OK;
}

static UArgs make_uargs(lise_ctx* c, int q, size_t off, int ns, int wb)
{
    UArgs u;
    u.L = c->L; u.W = Wbuf(c, wb);
    u.sA = S(c, q, RA) + off; u.sB = S(c, q, RB) + off; u.sC = S(c, q, RC) + off; u.sD = S(c, q, RD) + off;
    u.sE = S(c, q, RE) + off; u.sF = S(c, q, RF) + off; u.sG = S(c, q, RG) + off;
    u.Z = nullptr; u.eta_part = etabuf(c, wb); u.eta_fix = c->eta_fix; u.part = c->part[q];
    fill_common(c, u.ctab);
    u.neta = neta(c); u.dt = c->dt; u.hbarc = c->par.hbarc; u.ns = ns; u.G = c->G; u.order = 0; u.remove_phase = c->par.remove_phase;
    u.write_f = 1;
    return u;
}
static DArgs make_dargs(lise_ctx* c, int q, const cplx* Z, int ns)
{
    DArgs d;
    d.L = c->L; d.Z = Z; d.part = c->part[q]; fill_common(c, d.ctab); fill_stab(c, d.stab); d.ns = ns; d.G = c->G;
    return d;
}

static int zero_partials(lise_ctx* c, int q)
{
    CK(cudaMemsetAsync(c->part[q], 0, sizeof(double) * (size_t)c->G * LISE_NACC * c->L.nxyz, c->stream));
    return LISE_OK;
}

// part[q] += densities of the ns states in Z (all passes), on the context's stream
static int dens_chunk(lise_ctx* c, int q, const cplx* Z, int ns)
{
    if (c->ks.v5) TRY(launch_dens_yz(c, make_dargs(c, q, Z, ns)));
    else {
        UArgs u = make_uargs(c, q, 0, ns, 0);
        u.Z = Z;
        TRY(launch_update<0>(c, u, c->stream));
    }
    TRY(launch_dens_x(c, make_dargs(c, q, Z, ns)));
    return LISE_OK;
}
static int dens_accumulate(lise_ctx* c, int q, const cplx* Z)
{
    const size_t slen = (size_t)4 * c->L.nxyz;
    if (c->ks.v5) return c->nwf[q] > 0 ? dens_chunk(c, q, Z, c->nwf[q]) : LISE_OK;   // one launch pair per species
    for (int s0 = 0; s0 < c->nwf[q]; s0 += c->chunk) {
        const int ns = (c->nwf[q] - s0 < c->chunk) ? c->nwf[q] - s0 : c->chunk;
        TRY(dens_chunk(c, q, Z + s0 * slen, ns));
    }
    return LISE_OK;
}

static int reduce_partials(lise_ctx* c, int q)
{
    const size_t n = (size_t)LISE_NACC * c->L.nxyz;
    k_reduce_partials<<<nblk(n, 256), 256, 0, c->stream>>>(c->part[q], c->G, n, c->acc[q]);
    CKL();
    return LISE_OK;
}

// acc[q] = sum over this rank's partial buffers; then the sum over ranks through the hook (if any)
static int reduce_all(lise_ctx* c)
{
    TRY(reduce_partials(c, 0)); TRY(reduce_partials(c, 1));
    if (c->reduce_fn) {
        // the hook's contract names the CALLER's stream: bridge to it and back while the step runs on the internal one
        const bool bridge = c->user_stream_valid && c->stream != c->user_stream;
        if (bridge) { CK(cudaEventRecord(c->ev_fork, c->stream)); CK(cudaStreamWaitEvent(c->user_stream, c->ev_fork, 0)); }
        if (c->reduce_fn(c->reduce_user, c->acc[0], 2L * LISE_NACC * c->L.nxyz) != 0) {
            snprintf(c->err, sizeof(c->err), "reduce hook failed");
            return LISE_ECUDA;
        }
        if (bridge) { CK(cudaEventRecord(c->ev_join, c->user_stream)); CK(cudaStreamWaitEvent(c->stream, c->ev_join, 0)); }
    }
    return LISE_OK;
}

static int coulomb(lise_ctx* c, const double* np)
{
    const int nx = c->L.nx, ny = c->L.ny, nz = c->L.nz, P = c->P;
    const int T = 128;
    k_dft_pass_real<<<nblk((size_t)nx * ny * P, T), T, 0, c->stream>>>(np, c->cA1, c->tw, nx * ny, nz, P, 1, P); CKL();
    k_dft_pass<1><<<nblk((size_t)nx * P * P, T), T, 0, c->stream>>>(c->cA1, c->cA2, c->tw, nx, ny, P, P, P); CKL();
    k_dft_pass<1><<<nblk((size_t)P * P * P, T), T, 0, c->stream>>>(c->cA2, c->cA3, c->tw, 1, nx, P, P * P, P); CKL();
    k_coulomb_kernel_mult<<<nblk((size_t)P * P * P, 256), 256, 0, c->stream>>>(c->cA3, P, c->L.dx, c->Dc); CKL();
    k_dft_pass<-1><<<nblk((size_t)nx * P * P, T), T, 0, c->stream>>>(c->cA3, c->cA2, c->tw, 1, P, nx, P * P, P); CKL();
    k_dft_pass<-1><<<nblk((size_t)nx * ny * P, T), T, 0, c->stream>>>(c->cA2, c->cA1, c->tw, nx, P, ny, P, P); CKL();
    const double scale = c->par.e2 / ((double)P * P * P);
    k_dft_pass_final<<<nblk((size_t)nx * ny * nz, T), T, 0, c->stream>>>(c->cA1, c->phi, c->tw, nx * ny, P, nz, P, scale); CKL();
    return LISE_OK;
}

// potentials of both species from the reduced accumulators acc[0], acc[1]
// amp: amplitude of the external fields of Eq. 24 at the time this Hamiltonian belongs to (lise_set_external_amplitudes)
static int compute_potentials(lise_ctx* c, double amp)
{
    const int nx = c->L.nxyz;
    if (c->pc.coulomb) TRY(coulomb(c, c->acc[1] + (size_t)ACC_N * nx));
    k_grid_deriv<<<dim3(nblk(nx, 128), c->njobs1), 128, 0, c->stream>>>(c->L, c->jobs1, c->ctab[0], c->ctab[1], c->ctab[2]); CKL();
    ExtFields ext;
    ext.amp = amp;
    for (int q = 0; q < 2; ++q) { ext.u0[q] = c->uext[q]; ext.uvec[q] = c->vext[q]; }
    k_potentials<<<nblk(nx, 128), 128, 0, c->stream>>>(c->L, c->pc, ext, c->acc[0], c->acc[1], c->gtmp, c->phi,
                                                        c->dens[0], c->dens[1], c->pot[0], c->pot[1], c->geff[0], c->geff[1]); CKL();
    k_grid_deriv<<<dim3(nblk(nx, 128), c->njobs2), 128, 0, c->stream>>>(c->L, c->jobs2, c->ctab[0], c->ctab[1], c->ctab[2]); CKL();
    k_uloc<<<nblk(nx, 128), 128, 0, c->stream>>>(nx, c->pot[0], c->pot[1]); CKL();
    return LISE_OK;
}

// grid-only work between the barriers, timed as one class
static int grid_phase(lise_ctx* c, int reduce, double amp)
{
    prof_begin(c, PC_GRID);
    if (reduce) TRY(reduce_all(c));
    TRY(compute_potentials(c, amp));
    prof_end(c);
    return LISE_OK;
}

static int ensure_potentials(lise_ctx* c)
{
    if (c->pot_valid) return LISE_OK;
    TRY(grid_phase(c, 1, c->amp_now));              // the current wavefunctions y_n live at t_n
    c->pot_valid = 1;
    return LISE_OK;
}

// L637: psi_k <- psi_k / sqrt(<psi_k|psi_k>) for every state of slot `r` of both species (optional, lise_params.renormalize)
static int renormalize_slot(lise_ctx* c, int r)
{
    const size_t slen = (size_t)4 * c->L.nxyz;
    for (int q = 0; q < 2; ++q) {
        if (c->nwf[q] == 0) continue;
        k_state_norms<<<c->nwf[q], 256, 0, c->stream>>>(S(c, q, r), slen, c->L.dV, c->nrm); CKL();
        k_state_scale<<<dim3(nblk(slen, 256), c->nwf[q]), 256, 0, c->stream>>>(S(c, q, r), slen, c->nrm); CKL();
    }
    return LISE_OK;
}

static void rotate_f(lise_ctx* c)
{
    const int rc = c->role[RC], rd = c->role[RD], re = c->role[RE];
    c->role[RD] = rc; c->role[RE] = rd; c->role[RC] = re;
}

// one ABM predictor-modifier-corrector step (Eq. 78).
// plane5 kernels: software pipeline over chunks -- the DMMA-bound kernels (H-apply of chunk i + 1, densities of
// chunk i - 1) run on the context's stream while the HBM-bound update of chunk i runs on stream2; W and the eta
// partial sums are double-buffered.  Everything is joined back into the context's stream before returning.
static int abm_step(lise_ctx* c)
{
    const size_t slen = (size_t)4 * c->L.nxyz;
    TRY(ensure_potentials(c));                      // potentials of y_n
    const bool pipe = c->ks.v5 && c->overlap;
    for (int phase = 1; phase <= 2; ++phase) {
        TRY(zero_partials(c, 0)); TRY(zero_partials(c, 1));
        int i = 0;                                  // chunk counter across both species
        // densities of the new state: accumulated over groups of `dgroup` chunks (one launch pair per group), behind
        // the H-apply of the following chunk so that the update of the last chunk of the group overlaps it
        int pend_q = -1, pend_ns = 0, pend_chunks = 0; size_t pend_off = 0;
        auto flush_dens = [&](int last_chunk) -> int {
            if (pend_q < 0) return LISE_OK;
            if (pipe) CK(cudaStreamWaitEvent(c->stream, c->ev_u[last_chunk & 1], 0));
            TRY(dens_chunk(c, pend_q, (phase == 1 ? S(c, pend_q, RG) : S(c, pend_q, RB)) + pend_off, pend_ns));
            pend_q = -1; pend_ns = 0; pend_chunks = 0;
            return LISE_OK;
        };
        for (int q = 0; q < 2; ++q)
            for (int s0 = 0; s0 < c->nwf[q]; s0 += c->chunk, ++i) {
                const int ns = (c->nwf[q] - s0 < c->chunk) ? c->nwf[q] - s0 : c->chunk;
                const size_t off = s0 * slen;
                const int wb = pipe ? (i & 1) : 0;
                const cplx* X = (phase == 1 ? S(c, q, RA) : S(c, q, RG)) + off;
                if (pipe && i >= 2) CK(cudaStreamWaitEvent(c->stream, c->ev_u[wb], 0));   // W[wb], eta[wb] are free again
                TRY(apply_h_chunk(c, q, X, Wbuf(c, wb), etabuf(c, wb), ns));
                UArgs u = make_uargs(c, q, off, ns, wb);
                cudaStream_t su = pipe ? c->stream2 : c->stream;
                if (pipe) { CK(cudaEventRecord(c->ev_h[wb], c->stream)); CK(cudaStreamWaitEvent(c->stream2, c->ev_h[wb], 0)); }
                if (phase == 1) TRY(launch_update<1>(c, u, su)); else TRY(launch_update<2>(c, u, su));
                if (pipe) CK(cudaEventRecord(c->ev_u[wb], c->stream2));
                if (phase == 2 && c->par.renormalize) continue;    // densities of y_{n+1} follow the rescaling below
                if (c->ks.v5) {
                    if (pend_q >= 0 && (pend_q != q || pend_chunks >= c->dgroup)) TRY(flush_dens(i - 1));
                    if (pend_q < 0) { pend_q = q; pend_off = off; }
                    pend_ns += ns; pend_chunks += 1;
                } else {
                    TRY(launch_dens_x(c, make_dargs(c, q, (phase == 1 ? S(c, q, RG) : S(c, q, RB)) + off, ns)));
                }
            }
        TRY(flush_dens(i - 1));
        if (phase == 2 && c->par.renormalize) {
            if (pipe) for (int b = 0; b < 2; ++b) CK(cudaStreamWaitEvent(c->stream, c->ev_u[b], 0));   // all updates done
            TRY(renormalize_slot(c, RB));
            for (int q = 0; q < 2; ++q) {
                TRY(zero_partials(c, q));              // (the generic update kernels already added y/z parts of the unscaled state)
                if (c->nwf[q] > 0) TRY(dens_accumulate(c, q, S(c, q, RB)));
            }
        }
        if (phase == 1) TRY(grid_phase(c, 1, c->amp_next));   // potentials of the modifier m ~ y(t_{n+1}): fields at t_{n+1}
    }
    // y_{n+1} sits in B: A <-> B; f history shifts
    const int ra = c->role[RA]; c->role[RA] = c->role[RB]; c->role[RB] = ra;
    rotate_f(c);
    c->pot_valid = 0;                               // part[] now holds the densities of y_{n+1}
    return LISE_OK;
}

// T4(P) applied to y_n of every state: acc (slot F) = sum_{m<=4} (1/m!) [dt (H - eta)/(i hbar c)]^m y_n  (Eq. 77)
static int taylor4_all(lise_ctx* c, int write_f)
{
    const size_t slen = (size_t)4 * c->L.nxyz;
    for (int q = 0; q < 2; ++q)
        for (int s0 = 0; s0 < c->nwf[q]; s0 += c->chunk) {
            const int ns = (c->nwf[q] - s0 < c->chunk) ? c->nwf[q] - s0 : c->chunk;
            const size_t off = s0 * slen;
            for (int m = 1; m <= 4; ++m) {
                const cplx* X = (m == 1 ? S(c, q, RA) : S(c, q, RG)) + off;
                TRY(apply_h_chunk(c, q, X, Wbuf(c, 0), etabuf(c, 0), ns));
                UArgs u = make_uargs(c, q, off, ns, 0);
                u.order = m; u.write_f = write_f;
                TRY(launch_update<3>(c, u, c->stream));
            }
        }
    return LISE_OK;
}

// one start-up step: series expansion with predictor-corrector densities (Eqs. 75-77)
static int starter_step(lise_ctx* c)
{
    const size_t nacc = (size_t)LISE_NACC * c->L.nxyz;
    TRY(ensure_potentials(c));                      // H(t) from n(t); acc[] = accumulators of y_n
    for (int q = 0; q < 2; ++q)
        CK(cudaMemcpyAsync(c->acc0[q], c->acc[q], sizeof(double) * nacc, cudaMemcpyDeviceToDevice, c->stream));
    TRY(taylor4_all(c, 1));                         // psi_pre -> F, f_n -> C
    for (int q = 0; q < 2; ++q) {                   // n_cor = (n_pre + n(t)) / 2
        TRY(zero_partials(c, q));
        TRY(dens_accumulate(c, q, S(c, q, RF)));
    }
    TRY(reduce_all(c));
    for (int q = 0; q < 2; ++q) { k_average<<<nblk(nacc, 256), 256, 0, c->stream>>>(c->acc[q], c->acc0[q], nacc); CKL(); }
    TRY(compute_potentials(c, 0.5 * (c->amp_now + c->amp_next)));   // H_cor: fields averaged like the densities (B33)
    TRY(taylor4_all(c, 0));                         // y_{n+1} -> F
    if (c->par.renormalize) TRY(renormalize_slot(c, RF));
    for (int q = 0; q < 2; ++q) {
        TRY(zero_partials(c, q));
        TRY(dens_accumulate(c, q, S(c, q, RF)));
    }
    // A' = F (y_{n+1}), B' = A (y_n), F' = old B cleared (e = 0); f history shifts
    const int ra = c->role[RA], rb = c->role[RB], rf = c->role[RF];
    c->role[RA] = rf; c->role[RB] = ra; c->role[RF] = rb;
    rotate_f(c);
    for (int q = 0; q < 2; ++q)
        CK(cudaMemsetAsync(S(c, q, RF), 0, sizeof(cplx) * (size_t)c->nwf[q] * 4 * c->L.nxyz, c->stream));
    c->pot_valid = 0;
    return LISE_OK;
}

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
static int build_jobs(lise_ctx* c)
{
    const size_t nx = c->L.nxyz;
    std::vector<GJob> j1, j2;
    auto term = [](const double* in, int axis, int order, double sign) { GTerm t; t.in = in; t.axis = axis; t.order = order; t.sign = sign; return t; };
    for (int q = 0; q < 2; ++q) {
        const double* a = c->acc[q];
        double* g = c->gtmp + (size_t)q * GT_PER_Q * nx;
        GJob jb;
        // lap n
        jb.nterms = 3; jb.out = g + (size_t)GT_LAPN * nx;
        for (int i = 0; i < 3; ++i) jb.t[i] = term(a + (size_t)ACC_N * nx, i, 2, 1.0);
        j1.push_back(jb);
        // grad n
        for (int i = 0; i < 3; ++i) { jb.nterms = 1; jb.out = g + (size_t)(GT_GRADN + i) * nx; jb.t[0] = term(a + (size_t)ACC_N * nx, i, 1, 1.0); j1.push_back(jb); }
        // div J
        jb.nterms = 3; jb.out = g + (size_t)GT_DIVJ * nx;
        for (int i = 0; i < 3; ++i) jb.t[i] = term(a + (size_t)(ACC_J + i) * nx, i, 1, 1.0);
        j1.push_back(jb);
        // curl j, curl s: (curl v)_k = D_i v_j - D_j v_i, (k, i, j) cyclic
        for (int w = 0; w < 2; ++w) {
            const int src = w ? ACC_S : ACC_JC, dst = w ? GT_CURLS : GT_CURLJ;
            for (int k = 0; k < 3; ++k) {
                const int i = (k + 1) % 3, jx = (k + 2) % 3;
                jb.nterms = 2; jb.out = g + (size_t)(dst + k) * nx;
                jb.t[0] = term(a + (size_t)(src + jx) * nx, i, 1, 1.0);
                jb.t[1] = term(a + (size_t)(src + i) * nx, jx, 1, -1.0);
                j1.push_back(jb);
            }
        }
        // lap M
        jb.nterms = 3; jb.out = c->pot[q] + (size_t)P_LAPM * nx;
        for (int i = 0; i < 3; ++i) jb.t[i] = term(c->pot[q] + (size_t)P_M * nx, i, 2, 1.0);
        j2.push_back(jb);
    }
    c->njobs1 = (int)j1.size(); c->njobs2 = (int)j2.size();
    DM(c->jobs1, j1.size()); DM(c->jobs2, j2.size());
    CK(cudaMemcpy(c->jobs1, j1.data(), sizeof(GJob) * j1.size(), cudaMemcpyHostToDevice));
    CK(cudaMemcpy(c->jobs2, j2.data(), sizeof(GJob) * j2.size(), cudaMemcpyHostToDevice));
    return LISE_OK;
}

static int default_chunk(const lise_ctx* c)
{
    const double sbytes = 64.0 * c->L.nxyz;
    int nmax = c->nwf[0] > c->nwf[1] ? c->nwf[0] : c->nwf[1];
    int ch = (int)(255.0 * 1048576.0 / sbytes);      // W chunk of ~255 MB: measured flat optimum (170 .. 340 MB within 2 %)
    if (ch < c->G) ch = c->G;
    ch = (ch / c->G) * c->G;
    if (ch > nmax) ch = nmax;
    if (ch < 1) ch = 1;
    return ch;
}

// Coulomb work arrays (padded cube of side P = 3 max(N)); allocated when Coulomb is first switched on
static int alloc_coulomb(lise_ctx* c)
{
    if (c->tw) return LISE_OK;
    const Lattice& L = c->L;
    const int P = c->P;
    std::vector<double2> tw(P);
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int r = 0; r < P; ++r) { long double ph = 2.0L * pi * r / P; tw[r] = make_double2((double)cosl(ph), (double)-sinl(ph)); }
    DM(c->tw, P);
    CK(cudaMemcpy(c->tw, tw.data(), sizeof(double2) * P, cudaMemcpyHostToDevice));
    DM(c->cA1, (size_t)L.nx * L.ny * P); DM(c->cA2, (size_t)L.nx * P * P); DM(c->cA3, (size_t)P * P * P);
    return LISE_OK;
}

static int ctx_init(lise_ctx* c)
{
    const Lattice& L = c->L;
    const size_t nx = L.nxyz;
    // blocking and launch shapes
    c->R = (L.nx % 4 == 0 && L.ny % 4 == 0 && L.nz % 4 == 0) ? 4 : 2;
    c->mma = pick_kernels(L.nx, L.ny, L.nz, c->R, &c->ks, c->lop_mode) ? 1 : 0;
    if (!c->mma && !c->ks.name) {
        snprintf(c->err, sizeof(c->err), "no %s kernels were instantiated for a %d x %d x %d lattice",
                 c->lop_mode == LOP_FFT ? "fft" : "dmma", L.nx, L.ny, L.nz);
        return LISE_EUNSUPPORTED;
    }
    // the FFT kernels load their planes through TMA tensor maps: without the driver's encode entry point they cannot
    // run, so an automatic choice falls back to the generic kernels here, before anything is sized for the set
    if (c->mma && (c->ks.tma_h[0] || c->ks.tma_h[1]) && !resolve_encode_tiled()) {
        if (c->lop_mode == LOP_FFT) { snprintf(c->err, sizeof(c->err), "cuTensorMapEncodeTiled not available: the fft kernels cannot run"); return LISE_EUNSUPPORTED; }
        c->mma = pick_kernels(L.nx, L.ny, L.nz, c->R, &c->ks, LOP_DENSE) ? 1 : 0;
    }
    if (!c->mma) {
        const int ld = L.nz + 1;
        const int n1[2] = {L.ny, L.nx};
        for (int k = 0; k < 2; ++k) {
            const int npts = n1[k] * L.nz;
            int t = ((2 * npts / c->R + 31) / 32) * 32;
            if (t > 512) t = 512;
            if (t < 64) t = 64;
            c->ks.thr_h[k] = t;
            c->ks.smem_h[k] = sizeof(double2) * (size_t)(2 * (n1[k] + L.nz) + 8 * n1[k] * ld) + 64 * sizeof(double);
        }
        c->ks.thr_u = c->ks.thr_h[0]; c->ks.thr_d = c->ks.thr_h[1];
        c->ks.smem_u = sizeof(double2) * (size_t)(2 * (L.ny + L.nz) + 6 * L.ny * ld) + 64 * sizeof(double);
        c->ks.smem_d = sizeof(double2) * (size_t)(2 * L.nx + 6 * L.nx * ld);
    }
    const size_t lim = 227 * 1024;
    if (c->ks.smem_h[0] > lim || c->ks.smem_h[1] > lim || c->ks.smem_u > lim || c->ks.smem_d > lim) {
        snprintf(c->err, sizeof(c->err), "lattice planes too large for shared memory (%zu bytes needed, %zu available)",
                 c->ks.smem_h[0] > c->ks.smem_h[1] ? c->ks.smem_h[0] : c->ks.smem_h[1], lim);
        return LISE_EUNSUPPORTED;
    }
    TRY(set_attrs(c));
    int nsm = 148;
    { int dev = 0; if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev); if (nsm < 1) nsm = 148; }
    if (c->mma) {
        // plane-owner CTAs, one per SM: as many state groups as fit the SM count
        const int maxp = L.nx > L.ny ? L.nx : L.ny;
        c->G = nsm / maxp;
    } else {
        const int minp = L.nx < L.ny ? L.nx : L.ny;
        c->G = (2 * nsm + minp - 1) / minp;
    }
    if (c->G > LISE_MAXG) c->G = LISE_MAXG;
    if (c->G < 1) c->G = 1;
    c->chunk = default_chunk(c);
    const int nmax = c->nwf[0] > c->nwf[1] ? c->nwf[0] : c->nwf[1];

    // derivative tables
    for (int i = 0; i < 3; ++i) {
        std::vector<double2> t;
        host_ctab(c->n[i], L.dx, t);
        DM(c->ctab[i], t.size());
        CK(cudaMemcpy(c->ctab[i], t.data(), sizeof(double2) * t.size(), cudaMemcpyHostToDevice));
    }
    for (int i = 0; i < 3; ++i) {
        std::vector<double> t;
        host_stab(c->n[i], L.dx, t);
        DM(c->stab[i], t.size());
        CK(cudaMemcpy(c->stab[i], t.data(), sizeof(double) * t.size(), cudaMemcpyHostToDevice));
    }
    TRY(upload_rdft());
    {
        int lo = 0, hi = 0;
        CK(cudaDeviceGetStreamPriorityRange(&lo, &hi));
        CK(cudaStreamCreateWithPriority(&c->stream2, cudaStreamNonBlocking, lo));
        CK(cudaStreamCreateWithPriority(&c->streamH, cudaStreamNonBlocking, hi));
        CK(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
    }
    for (int i = 0; i < 2; ++i) {
        CK(cudaEventCreateWithFlags(&c->ev_h[i], cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&c->ev_u[i], cudaEventDisableTiming));
    }
    c->overlap = 1;
    c->dgroup = 8;
    // state slots and scratch
    for (int q = 0; q < 2; ++q)
        for (int s = 0; s < LISE_NSLOT; ++s) {
            DM(c->slot[q][s], (size_t)c->nwf[q] * 4 * nx);
            CK(cudaMemset(c->slot[q][s], 0, sizeof(cplx) * (size_t)c->nwf[q] * 4 * nx));
        }
    for (int s = 0; s < LISE_NSLOT; ++s) c->role[s] = s;
    c->wcap = nmax < 256 ? (nmax > 0 ? nmax : 1) : 256;     // largest chunk lise_set_chunk accepts
    if (c->wcap < c->chunk) c->wcap = c->chunk;
    DM(c->W, (size_t)2 * c->wcap * 4 * nx);
    DM(c->eta_part, (size_t)2 * c->wcap * L.ny * 2);
    DM(c->eta_fix, (size_t)c->wcap);
    for (int q = 0; q < 2; ++q) {
        DM(c->part[q], (size_t)LISE_MAXG * LISE_NACC * nx);
        CK(cudaMemset(c->part[q], 0, sizeof(double) * (size_t)LISE_MAXG * LISE_NACC * nx));
        DM(c->acc0[q], LISE_NACC * nx);
        DM(c->dens[q], 14 * nx); DM(c->pot[q], LISE_NPOT * nx); DM(c->geff[q], nx);
        CK(cudaMemset(c->pot[q], 0, sizeof(double) * LISE_NPOT * nx));
    }
    DM(c->acc[0], 2 * LISE_NACC * nx);                       // both species contiguous: one all-reduce
    c->acc[1] = c->acc[0] + (size_t)LISE_NACC * nx;
    DM(c->gtmp, 2 * GT_PER_Q * nx);
    DM(c->phi, nx);
    CK(cudaMemset(c->phi, 0, sizeof(double) * nx));
    TRY(build_jobs(c));
    // Coulomb
    int nm = L.nx; if (L.ny > nm) nm = L.ny; if (L.nz > nm) nm = L.nz;
    c->P = 3 * nm; c->Dc = sqrt(3.0) * L.dx * nm;
    if (c->par.coulomb) TRY(alloc_coulomb(c));
    c->eblocks = 64;
    DM(c->ebuf, c->eblocks * 6);
    DM(c->mbuf, c->eblocks * 16);
    DM(c->nrm, nmax > 0 ? nmax : 1);
    DM(c->ovl, (size_t)(nmax > 0 ? nmax : 1) * 4);
    return LISE_OK;
}

static thread_local char t_create_err[288] = "";   // message of this thread's last failed lise_create (there is no context to ask)
static int create_impl(int nx, int ny, int nz, double dx, double dt, int nwf_n, int nwf_p, int lop_mode, lise_ctx** out)
{
    if (!out) return LISE_EINVAL;
    *out = nullptr;
    t_create_err[0] = 0;
    if (nx < 2 || ny < 2 || nz < 2 || ((nx | ny | nz) & 1) || !(dx > 0.0) || nwf_n < 0 || nwf_p < 0) return LISE_EINVAL;
    if ((long long)nx * ny * nz > (1LL << 26)) return LISE_EUNSUPPORTED;
    lise_ctx* c = new (std::nothrow) lise_ctx();
    if (!c) return LISE_ENOMEM;
    memset(c, 0, sizeof(*c));
    c->allocs = new std::vector<void*>();
    c->prof_ev = new std::vector<cudaEvent_t>();
    c->prof_cls = new std::vector<int>();
    c->L.nx = nx; c->L.ny = ny; c->L.nz = nz; c->L.nxyz = nx * ny * nz; c->L.dx = dx; c->L.dV = dx * dx * dx;
    c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
    c->dt = dt; c->nwf[0] = nwf_n; c->nwf[1] = nwf_p;
    lise_default_params(&c->par);
    if (nwf_p == 0) c->par.coulomb = 0;
    set_physconst(c);
    c->stream = 0;
    c->have[0] = (nwf_n == 0); c->have[1] = (nwf_p == 0);
    c->lop_mode = lop_mode;
    c->amp_now = c->amp_next = 1.0;
    int rc = ctx_init(c);
    if (rc != LISE_OK) {
        snprintf(t_create_err, sizeof(t_create_err), "lise_create: %s", c->err);
        lise_destroy(c);
        return rc;
    }
    *out = c;
    return LISE_OK;
}
extern "C" int lise_create(int nx, int ny, int nz, double dx, double dt, int nwf_n, int nwf_p, lise_ctx** out)
{
    return guarded([&] { return create_impl(nx, ny, nz, dx, dt, nwf_n, nwf_p, LOP_AUTO, out); });
}
extern "C" int lise_create_with_line_operator(int nx, int ny, int nz, double dx, double dt, int nwf_n, int nwf_p,
                                              const char* line_operator, lise_ctx** out)
{
    int mode = LOP_AUTO;
    if (line_operator && strcmp(line_operator, "auto") != 0) {
        if (!strcmp(line_operator, "fft")) mode = LOP_FFT;
        else if (!strcmp(line_operator, "dmma")) mode = LOP_DMMA;
        else if (!strcmp(line_operator, "dense")) mode = LOP_DENSE;
        else { if (out) *out = nullptr; snprintf(t_create_err, sizeof(t_create_err), "lise_create: unknown line operator \"%.40s\"", line_operator); return LISE_EINVAL; }
    }
    return guarded([&] { return create_impl(nx, ny, nz, dx, dt, nwf_n, nwf_p, mode, out); });
}

extern "C" void lise_destroy(lise_ctx* c)
{
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    if (c->stream2) { cudaStreamSynchronize(c->stream2); cudaStreamDestroy(c->stream2); }
    if (c->streamH) { cudaStreamSynchronize(c->streamH); cudaStreamDestroy(c->streamH); }
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    for (int i = 0; i < 2; ++i) { if (c->ev_h[i]) cudaEventDestroy(c->ev_h[i]); if (c->ev_u[i]) cudaEventDestroy(c->ev_u[i]); }
    if (c->allocs) {
        for (void* p : *c->allocs) cudaFree(p);
        delete c->allocs;
    }
    if (c->prof_ev) { for (cudaEvent_t e : *c->prof_ev) cudaEventDestroy(e); delete c->prof_ev; }
    delete c->prof_cls;
    delete c;
}

extern "C" int lise_set_params(lise_ctx* c, const lise_params* p)
{
    if (!c || !p) return LISE_EINVAL;
    c->par = *p;
    if (c->par.coulomb) { const int rc = guarded([&] { return alloc_coulomb(c); }); if (rc != LISE_OK) return rc; }
    set_physconst(c);
    c->pot_valid = 0;
    return LISE_OK;
}

extern "C" int lise_set_stream(lise_ctx* c, void* s)
{
    if (!c) return LISE_EINVAL;
    c->stream = (cudaStream_t)s;
    return LISE_OK;
}

extern "C" int lise_set_dt(lise_ctx* c, double dt)
{
    if (!c) return LISE_EINVAL;
    c->dt = dt; c->step = 0; c->since = 0;
    return LISE_OK;
}

extern "C" int lise_set_chunk(lise_ctx* c, int n)
{
    if (!c) return LISE_EINVAL;
    if (n <= 0) c->chunk = default_chunk(c);
    else c->chunk = n > c->wcap ? c->wcap : n;
    return LISE_OK;
}

extern "C" int lise_set_overlap(lise_ctx* c, int enable)
{
    if (!c) return LISE_EINVAL;
    c->overlap = enable ? 1 : 0;
    return LISE_OK;
}

extern "C" int lise_set_density_group(lise_ctx* c, int nchunks)
{
    if (!c) return LISE_EINVAL;
    c->dgroup = nchunks > 0 ? nchunks : 8;
    return LISE_OK;
}

extern "C" int lise_set_wavefunctions(lise_ctx* c, int q, const void* psi_dev)
{
    if (!c || q < 0 || q > 1 || (!psi_dev && c->nwf[q] > 0)) return LISE_EINVAL;
    const size_t bytes = sizeof(cplx) * (size_t)c->nwf[q] * 4 * c->L.nxyz;
    if (c->nwf[q] > 0) CK(cudaMemcpyAsync(S(c, q, RA), psi_dev, bytes, cudaMemcpyDeviceToDevice, c->stream));
    TRY(zero_partials(c, q));
    if (c->nwf[q] > 0) TRY(dens_accumulate(c, q, S(c, q, RA)));
    c->have[q] = 1; c->pot_valid = 0; c->step = 0; c->since = 0; c->time = 0.0;
    return LISE_OK;
}

extern "C" int lise_get_wavefunctions(lise_ctx* c, int q, void* psi_dev)
{
    if (!c || q < 0 || q > 1 || (!psi_dev && c->nwf[q] > 0)) return LISE_EINVAL;
    if (!c->have[q]) { snprintf(c->err, sizeof(c->err), "wavefunctions of species %d not set", q); return LISE_ESTATE; }
    const size_t bytes = sizeof(cplx) * (size_t)c->nwf[q] * 4 * c->L.nxyz;
    if (c->nwf[q] > 0) CK(cudaMemcpyAsync(psi_dev, S(c, q, RA), bytes, cudaMemcpyDeviceToDevice, c->stream));
    return LISE_OK;
}

extern "C" int lise_upload_wavefunctions(lise_ctx* c, int q, const void* psi_host, int keep_history)
{
    if (!c || q < 0 || q > 1 || (!psi_host && c->nwf[q] > 0)) return LISE_EINVAL;
    if (keep_history && !c->have[q]) { snprintf(c->err, sizeof(c->err), "no history to keep for species %d", q); return LISE_ESTATE; }
    const size_t bytes = sizeof(cplx) * (size_t)c->nwf[q] * 4 * c->L.nxyz;
    if (c->nwf[q] > 0) CK(cudaMemcpyAsync(S(c, q, RA), psi_host, bytes, cudaMemcpyHostToDevice, c->stream));
    TRY(zero_partials(c, q));
    if (c->nwf[q] > 0) TRY(dens_accumulate(c, q, S(c, q, RA)));
    c->have[q] = 1; c->pot_valid = 0;
    if (!keep_history) { c->step = 0; c->since = 0; c->time = 0.0; }
    return LISE_OK;
}

extern "C" int lise_download_wavefunctions(lise_ctx* c, int q, void* psi_host)
{
    if (!c || q < 0 || q > 1 || (!psi_host && c->nwf[q] > 0)) return LISE_EINVAL;
    if (!c->have[q]) { snprintf(c->err, sizeof(c->err), "wavefunctions of species %d not set", q); return LISE_ESTATE; }
    const size_t bytes = sizeof(cplx) * (size_t)c->nwf[q] * 4 * c->L.nxyz;
    if (c->nwf[q] > 0) CK(cudaMemcpyAsync(psi_host, S(c, q, RA), bytes, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return LISE_OK;
}

extern "C" int lise_set_reduce_hook(lise_ctx* c, lise_reduce_fn fn, void* user)
{
    if (!c) return LISE_EINVAL;
    c->reduce_fn = fn; c->reduce_user = user;
    c->pot_valid = 0;
    return LISE_OK;
}

static int need_both(lise_ctx* c)
{
    if (!c->have[0] || !c->have[1]) { snprintf(c->err, sizeof(c->err), "set the wavefunctions of both species first"); return LISE_ESTATE; }
    return LISE_OK;
}

extern "C" int lise_densities(lise_ctx* c, int q, double* out14_dev)
{
    if (!c || q < 0 || q > 1 || !out14_dev) return LISE_EINVAL;
    TRY(need_both(c));
    TRY(ensure_potentials(c));
    CK(cudaMemcpyAsync(out14_dev, c->dens[q], sizeof(double) * 14 * (size_t)c->L.nxyz, cudaMemcpyDeviceToDevice, c->stream));
    return LISE_OK;
}

extern "C" int lise_potentials(lise_ctx* c, int q, double* out14_dev)
{
    if (!c || q < 0 || q > 1 || !out14_dev) return LISE_EINVAL;
    TRY(need_both(c));
    TRY(ensure_potentials(c));
    CK(cudaMemcpyAsync(out14_dev, c->pot[q], sizeof(double) * 14 * (size_t)c->L.nxyz, cudaMemcpyDeviceToDevice, c->stream));
    return LISE_OK;
}

extern "C" int lise_apply_h(lise_ctx* c, int q, const void* in_dev, void* out_dev, int nstates)
{
    if (!c || q < 0 || q > 1 || nstates < 0 || (nstates > 0 && (!in_dev || !out_dev))) return LISE_EINVAL;
    if (nstates == 0) return LISE_OK;                // empty input: nothing to do, the pointers may be null
    TRY(need_both(c));
    TRY(ensure_potentials(c));
    const size_t slen = (size_t)4 * c->L.nxyz;
    const int ch = c->chunk;                       // eta_part scratch is sized for wcap >= chunk states
    for (int s0 = 0; s0 < nstates; s0 += ch) {
        const int ns = (nstates - s0 < ch) ? nstates - s0 : ch;
        TRY(apply_h_chunk(c, q, (const cplx*)in_dev + s0 * slen, (cplx*)out_dev + s0 * slen, etabuf(c, 0), ns));
    }
    return LISE_OK;
}

static int step_impl(lise_ctx* c, int nsteps)
{
    if (!c || nsteps < 0) return LISE_EINVAL;
    TRY(need_both(c));
    // overlap on: fork from the caller's stream into the internal high-priority stream, join at the end
    cudaStream_t user = c->stream;
    const bool fork = c->ks.v5 && c->overlap && nsteps > 0;
    if (fork) {
        CK(cudaEventRecord(c->ev_fork, user));
        CK(cudaStreamWaitEvent(c->streamH, c->ev_fork, 0));
        c->stream = c->streamH; c->user_stream = user; c->user_stream_valid = 1;
    }
    int rc = LISE_OK;
    for (int s = 0; s < nsteps && rc == LISE_OK; ++s) {
        rc = (c->since < 3) ? starter_step(c) : abm_step(c);
        if (rc == LISE_OK) { c->step += 1; c->since += 1; c->time += c->dt; }
    }
    if (fork) {
        c->stream = user; c->user_stream_valid = 0;
        CK(cudaEventRecord(c->ev_join, c->streamH));
        CK(cudaStreamWaitEvent(user, c->ev_join, 0));
    }
    return rc;
}
extern "C" int lise_step(lise_ctx* c, int nsteps)
{
    return guarded([&] { return step_impl(c, nsteps); });
}

static int observables_impl(lise_ctx* c, lise_observables_t* o)
{
    if (!c || !o) return LISE_EINVAL;
    TRY(need_both(c));
    TRY(ensure_potentials(c));
    k_energy<<<c->eblocks, 256, 0, c->stream>>>(c->L, c->pc, c->acc[0], c->acc[1], c->gtmp, c->phi, c->geff[0], c->geff[1], c->ebuf); CKL();
    std::vector<double> eb(c->eblocks * 6);
    CK(cudaMemcpyAsync(eb.data(), c->ebuf, sizeof(double) * eb.size(), cudaMemcpyDeviceToHost, c->stream));
    double nd = 0.0, od = 0.0;
    for (int q = 0; q < 2; ++q) {
        const int nw = c->nwf[q];
        if (nw == 0) continue;
        k_overlaps<<<dim3(nw, 4), 256, 0, c->stream>>>(S(c, q, RA), nw, 4 * c->L.nxyz, c->L.dV, c->ovl); CKL();
        std::vector<double2> ov((size_t)nw * 4);
        CK(cudaMemcpyAsync(ov.data(), c->ovl, sizeof(double2) * ov.size(), cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        const int ds[4] = {0, 1, 2, nw / 2};
        for (int k = 0; k < nw; ++k) {
            const double dn = fabs(ov[(size_t)k * 4].x - 1.0);
            if (dn > nd) nd = dn;
            for (int t = 1; t < 4; ++t) {
                if ((k + ds[t]) % nw == k) continue;
                const double m = hypot(ov[(size_t)k * 4 + t].x, ov[(size_t)k * 4 + t].y);
                if (m > od) od = m;
            }
        }
    }
    CK(cudaStreamSynchronize(c->stream));
    double e[6] = {0, 0, 0, 0, 0, 0};
    for (int b = 0; b < c->eblocks; ++b) for (int k = 0; k < 6; ++k) e[k] += eb[b * 6 + k];
    o->e_kin = e[0]; o->e_skyrme = e[1]; o->e_coul = e[2]; o->e_pair = e[3];
    o->energy = e[0] + e[1] + e[2] + e[3];
    o->n_neutron = e[4]; o->n_proton = e[5];
    o->norm_defect = nd; o->ortho_defect = od;
    o->time = c->time; o->step = c->step;
    return LISE_OK;
}
extern "C" int lise_observables(lise_ctx* c, lise_observables_t* o)
{
    return guarded([&] { return observables_impl(c, o); });
}

extern "C" int lise_set_time(lise_ctx* c, double time, long step)
{
    if (!c || step < 0) return LISE_EINVAL;
    c->time = time; c->step = step;
    return LISE_OK;
}

extern "C" int lise_boost(lise_ctx* c, int q, const double* chi_dev)
{
    if (!c || q < 0 || q > 1 || !chi_dev) return LISE_EINVAL;
    if (!c->have[q]) { snprintf(c->err, sizeof(c->err), "wavefunctions of species %d not set", q); return LISE_ESTATE; }
    if (c->nwf[q] > 0) {
        k_boost<<<dim3(nblk(c->L.nxyz, 128), 4, c->nwf[q]), 128, 0, c->stream>>>(S(c, q, RA), chi_dev, c->L.nxyz); CKL();
    }
    TRY(zero_partials(c, q));
    if (c->nwf[q] > 0) TRY(dens_accumulate(c, q, S(c, q, RA)));
    c->pot_valid = 0; c->since = 0;
    return LISE_OK;
}

extern "C" int lise_set_external_fields(lise_ctx* c, int q, const double* u0_dev, const double* uvec_dev)
{
    if (!c || q < 0 || q > 1) return LISE_EINVAL;
    const size_t nx = c->L.nxyz;
    // the buffers are allocated once and kept; a NULL argument switches the field off
    if (u0_dev) {
        if (!c->uext_buf[q]) DM(c->uext_buf[q], nx);
        CK(cudaMemcpyAsync(c->uext_buf[q], u0_dev, sizeof(double) * nx, cudaMemcpyDeviceToDevice, c->stream));
    }
    if (uvec_dev) {
        if (!c->vext_buf[q]) DM(c->vext_buf[q], 3 * nx);
        CK(cudaMemcpyAsync(c->vext_buf[q], uvec_dev, sizeof(double) * 3 * nx, cudaMemcpyDeviceToDevice, c->stream));
    }
    c->uext[q] = u0_dev ? c->uext_buf[q] : nullptr;
    c->vext[q] = uvec_dev ? c->vext_buf[q] : nullptr;
    c->pot_valid = 0;
    return LISE_OK;
}

extern "C" int lise_set_external_amplitudes(lise_ctx* c, double f_now, double f_next)
{
    if (!c || !(fabs(f_now) < INFINITY) || !(fabs(f_next) < INFINITY)) return LISE_EINVAL;
    c->amp_now = f_now; c->amp_next = f_next;
    c->pot_valid = 0;                               // the potentials of y_n carry f_now
    return LISE_OK;
}

extern "C" int lise_set_frame(lise_ctx* c, const double* v_cm, const double* omega, const double* origin)
{
    if (!c) return LISE_EINVAL;
    for (int i = 0; i < 3; ++i) {
        c->pc.vcm[i] = v_cm ? v_cm[i] : 0.0; c->pc.omega[i] = omega ? omega[i] : 0.0; c->pc.origin[i] = origin ? origin[i] : 0.0;
    }
    c->pot_valid = 0;
    return LISE_OK;
}

static int observables_ext_impl(lise_ctx* c, lise_observables_ext_t* o)
{
    if (!c || !o) return LISE_EINVAL;
    TRY(need_both(c));
    TRY(ensure_potentials(c));
    ExtFields ext;
    ext.amp = c->amp_now;
    for (int q = 0; q < 2; ++q) { ext.u0[q] = c->uext[q]; ext.uvec[q] = c->vext[q]; }
    const int nb = c->eblocks;
    k_moments1<<<nb, 256, 0, c->stream>>>(c->L, c->pc, ext, c->dens[0], c->dens[1], c->pot[0], c->pot[1], c->mbuf); CKL();
    std::vector<double> hb((size_t)nb * 16);
    CK(cudaMemcpyAsync(hb.data(), c->mbuf, sizeof(double) * hb.size(), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    double m[16];
    for (int k = 0; k < 16; ++k) { m[k] = 0.0; for (int b = 0; b < nb; ++b) m[k] += hb[(size_t)b * 16 + k]; }
    const double Nn = m[0], Np = m[1], A = Nn + Np;
    for (int i = 0; i < 3; ++i) {
        o->rcm_n[i] = Nn > 0.0 ? m[2 + i] / Nn : 0.0;
        o->rcm_p[i] = Np > 0.0 ? m[5 + i] / Np : 0.0;
        o->rcm[i] = A > 0.0 ? (m[2 + i] + m[5 + i]) / A : 0.0;
    }
    o->delta_n = Nn > 0.0 ? m[11] / Nn : 0.0;
    o->delta_p = Np > 0.0 ? m[12] / Np : 0.0;
    o->e_coll = m[13];
    o->e_ext = m[14];
    // Eq. 27: v_cm = hbar int j d^3r / (m A); hbar / m = 2 (hbar^2 / 2m) / (hbar c) in units of c.  Eq. 41: (1/2) m A v_cm^2
    double j2 = 0.0;
    for (int i = 0; i < 3; ++i) { o->v_cm[i] = A > 0.0 ? 2.0 * c->par.hbar2_2m / c->par.hbarc * m[8 + i] / A : 0.0; j2 += m[8 + i] * m[8 + i]; }
    o->e_cm = A > 0.0 ? c->par.hbar2_2m * j2 / A : 0.0;
    k_moments2<<<nb, 256, 0, c->stream>>>(c->L, c->dens[0], c->dens[1], o->rcm[0], o->rcm[1], o->rcm[2], c->mbuf); CKL();
    CK(cudaMemcpyAsync(hb.data(), c->mbuf, sizeof(double) * (size_t)nb * 8, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    double qm[8];
    for (int k = 0; k < 8; ++k) { qm[k] = 0.0; for (int b = 0; b < nb; ++b) qm[k] += hb[(size_t)b * 8 + k]; }
    o->q20 = qm[0]; o->q30 = qm[1]; o->q40 = qm[2];
    o->q21[0] = qm[3]; o->q21[1] = qm[4]; o->q22[0] = qm[5]; o->q22[1] = qm[6];
    return LISE_OK;
}
extern "C" int lise_observables_ext(lise_ctx* c, lise_observables_ext_t* o)
{
    return guarded([&] { return observables_ext_impl(c, o); });
}

extern "C" int lise_profile(lise_ctx* c, int enable)
{
    if (!c) return LISE_EINVAL;
    CK(cudaStreamSynchronize(c->stream));
    c->prof = enable ? 1 : 0; c->prof_n = 0;
    return LISE_OK;
}

extern "C" int lise_profile_read(lise_ctx* c, double* ms, long* counts)
{
    if (!c || !ms || !counts) return LISE_EINVAL;
    CK(cudaStreamSynchronize(c->stream));
    for (int k = 0; k < PC_NCLASS; ++k) { ms[k] = 0.0; counts[k] = 0; }
    for (int i = 0; i < c->prof_n; ++i) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, (*c->prof_ev)[2 * i], (*c->prof_ev)[2 * i + 1]));
        ms[(*c->prof_cls)[i]] += t; counts[(*c->prof_cls)[i]] += 1;
    }
    c->prof_n = 0;
    return LISE_OK;
}

extern "C" int lise_measure_fp64_peak(void* stream, double seconds, double* tflops_host, double* sm_mhz_host)
{
    if (!tflops_host || !(seconds > 0.0)) return LISE_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return LISE_ECUDA;
    double* out = nullptr;
    const int blocks = nsm * 8, threads = 256, iters = 4096;
    if (cudaMalloc(&out, sizeof(double) * blocks * threads) != cudaSuccess) return LISE_ENOMEM;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const double flop = 2.0 * PEAK_CHAINS * (double)iters * blocks * threads;
    double best = 0.0, total_ms = 0.0;
    int rc = LISE_OK;
    for (int rep = 0; rep < 100000 && total_ms < seconds * 1e3; ++rep) {   // sustained: keep the pipe busy for `seconds`
        cudaEventRecord(e0, st);
        for (int k = 0; k < 8; ++k) k_dfma_peak<<<blocks, threads, 0, st>>>(out, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = LISE_ECUDA; break; }
        float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
        total_ms += ms;
        const double tf = 8.0 * flop / (ms * 1e-3) * 1e-12;
        if (total_ms > 0.5 * seconds * 1e3 && tf > best) best = tf;      // the second half: under sustained load
        if (rep == 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    *tflops_host = best;
    if (sm_mhz_host) *sm_mhz_host = 0.0;
    return rc;
}

// host-only: the block-diagonalised tables of a line of n points (no CUDA call; tests pin them against Eqs. 49-50)
extern "C" int lise_line_operator_tables(int n, double dx, double* tab_host, int cap, int* dims_host)
{
    if (n < 4 || n % 4 != 0 || !(dx > 0.0) || !dims_host) return LISE_EINVAL;
    const LOpDims D = lop_dims(n);
    dims_host[0] = D.H; dims_host[1] = D.R; dims_host[2] = D.J; dims_host[3] = D.ND; dims_host[4] = D.TABSZ;
    if (!tab_host) return LISE_OK;
    if (cap < D.TABSZ) return LISE_EINVAL;
    std::vector<double> t;
    host_stab(n, dx, t);
    memcpy(tab_host, t.data(), sizeof(double) * t.size());
    return LISE_OK;
}

// host-only: fp64 instruction counts of the generated FFT codelets for a real line of n points (0, 0 if none)
extern "C" int lise_line_operator_cost(int n, int* inner_ops_host, int* outer_ops_host)
{
    if (!inner_ops_host || !outer_ops_host) return LISE_EINVAL;
    *inner_ops_host = 0; *outer_ops_host = 0;
    switch (n) {
#define X(N_) case N_: *inner_ops_host = LineCodelet<N_>::OPS_INNER; *outer_ops_host = LineCodelet<N_>::OPS_OUTER; break;
    X(4) X(6) X(8) X(10) X(12) X(16) X(20) X(24) X(32) X(40)
#undef X
    default: break;
    }
    return LISE_OK;
}

extern "C" const char* lise_line_operator(const lise_ctx* c) { return c ? c->ks.name : "none"; }

extern "C" long lise_launch_count(const lise_ctx* c) { return c ? c->launches : 0; }
extern "C" long long lise_device_bytes(const lise_ctx* c) { return c ? c->bytes : 0; }

extern "C" const char* lise_strerror(int code)
{
    switch (code) {
    case LISE_OK: return "ok";
    case LISE_EINVAL: return "invalid argument";
    case LISE_ESTATE: return "wavefunctions not set";
    case LISE_ECUDA: return "CUDA error";
    case LISE_ENOMEM: return "out of device memory";
    case LISE_EUNSUPPORTED: return "unsupported lattice size";
    default: return "unknown error";
    }
}
extern "C" const char* lise_last_error(const lise_ctx* c) { return c ? c->err : (t_create_err[0] ? t_create_err : g_noctx); }
