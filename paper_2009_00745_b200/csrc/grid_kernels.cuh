// grid_kernels.cuh -- grid-only work between the two global barriers of a time step:
// density reduction, lattice derivatives of real fields, mean-field / pairing potentials (Skyrme, SeaLL1), Coulomb,
// energy, the observables of Eqs. 37-41, and the small whole-state utilities (boost, renormalisation).
// All fields are Nxyz doubles; the work is tiny next to the per-state kernels, so these kernels are
// written for clarity and launch count, not for peak throughput.
#pragma once
#include "common.cuh"

struct PhysConst {
    double h2m, e2, hbarc, gamma, a, Kc;
    double Cn[2], Cg[2], Cd[2], Ct[2], CJ[2], g0[2];      // couplings of Eq. 9 by isospin t = 0, 1; bare pairing couplings by species
    double alpha, mu[2], ecut;                           // Eq. 8 (density-dependent g0), Eq. 20 (spherical cutoff)
    double sa[3], sb[3], sc[3];                          // Eq. 10: SeaLL1 volume coefficients
    double vcm[3], omega[3], origin[3];                  // Eqs. 26, 36: frame velocity (units of c), angular velocity (c / fm), its origin
    int coulomb, rearr, functional, cutoff;
};
// external fields of Eq. 24 per species (device pointers, NULL = none): scalar U0 [Nxyz], vector Uvec [3][Nxyz]
struct ExtFields { const double* u0[2]; const double* uvec[2]; double amp; };   // amp: amplitude f(t) on both profiles

// acc[f][r] = sum_g part[g][f][r] in fixed order (deterministic)
__global__ void k_reduce_partials(const double* __restrict__ part, int G, size_t n, double* __restrict__ acc)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double s = 0.0;
    for (int g = 0; g < G; ++g) s += part[(size_t)g * n + i];
    acc[i] = s;
}

__global__ void k_average(double* __restrict__ a, const double* __restrict__ b, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = 0.5 * (a[i] + b[i]);
}

// out = sum_t sign_t * D^{(order_t)}_{axis_t} in_t   (up to 3 terms; lap, div, curl components, grad)
struct GTerm { const double* in; int axis, order; double sign; };
struct GJob { GTerm t[3]; int nterms; double* out; };

__global__ void k_grid_deriv(Lattice L, const GJob* __restrict__ jobs,
                             const double2* __restrict__ ct0, const double2* __restrict__ ct1, const double2* __restrict__ ct2)
{
    const GJob jb = jobs[blockIdx.y];
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= L.nxyz) return;
    const int iz = r % L.nz, iy = (r / L.nz) % L.ny, ix = r / (L.nz * L.ny);
    double s = 0.0;
    for (int t = 0; t < jb.nterms; ++t) {
        const GTerm tm = jb.t[t];
        int N, n, stride; const double2* ct;
        if (tm.axis == 0)      { N = L.nx; n = ix; stride = L.ny * L.nz; ct = ct0; }
        else if (tm.axis == 1) { N = L.ny; n = iy; stride = L.nz; ct = ct1; }
        else                   { N = L.nz; n = iz; stride = 1; ct = ct2; }
        const double* line = tm.in + (r - n * stride);
        double acc = 0.0;
        for (int m = 0; m < N; ++m) {
            const double2 c = ct[N + n - m];
            acc = fma(tm.order == 1 ? c.x : c.y, line[m * stride], acc);
        }
        s += tm.sign * acc;
    }
    jb.out[r] = s;
}

// gtmp layout per species q (11 fields): 0 lap n, 1..3 grad n, 4 div J, 5..7 curl j, 8..10 curl s
#define GT_PER_Q 11
enum { GT_LAPN = 0, GT_GRADN = 1, GT_DIVJ = 4, GT_CURLJ = 5, GT_CURLS = 8 };

// ------------------------------------------------------------------------------------------------
// The functional at one lattice point, in the ISOSPIN basis t = 0 (isoscalar), 1 (isovector) in which Eq. 9 is
// written.  eps = sum_t [ Cn n_t^2 + Cg n_t^2 n_0^gamma + Cd n_t lap n_t + Ct (n_t tau_t - j_t^2)
//                         + CJ (n_t div J_t + s_t . curl j_t) ]  (+ SeaLL1 volume term, Eq. 10),
// and every mean field is the partial derivative of eps with respect to the density it multiplies
// (H = dE / d psi^+), taken here term by term in t and rotated to the species basis at the end:
//   F_q = F_0 + xi_q F_1,  xi_n = +1, xi_p = -1  (d n_0 / d n_q = 1, d n_1 / d n_q = xi_q).
// ------------------------------------------------------------------------------------------------
struct IsoPoint {
    double n[2], tau[2], lapn[2], divJ[2];
    double j[2][3], s[2][3], gradn[2][3], curlj[2][3], curls[2][3];
};
__device__ __forceinline__ double pow_or_zero(double x, double p) { return x > 0.0 ? pow(x, p) : 0.0; }

// SeaLL1 volume energy (Eq. 10): sum_j F_j(n0) beta^(2j), F_j = a_j n0^(5/3) + b_j n0^2 + c_j n0^(7/3), beta = n1 / n0
// (reading B29).  Returns eps and its partial derivatives with respect to n0 and n1.
__device__ __forceinline__ void seall1_volume(const PhysConst& pc, double n0, double n1, double& eps, double& d0, double& d1)
{
    eps = d0 = d1 = 0.0;
    if (!(n0 > 0.0)) return;
    const double c13 = cbrt(n0), p53 = n0 * c13 * c13, p73 = n0 * n0 * c13, beta = n1 / n0, b2 = beta * beta;
    double bpow = 1.0;                                    // beta^(2j)
#pragma unroll
    for (int jx = 0; jx < 3; ++jx) {
        const double F = pc.sa[jx] * p53 + pc.sb[jx] * n0 * n0 + pc.sc[jx] * p73;
        const double dF = (5.0 / 3.0 * pc.sa[jx] * p53 + 2.0 * pc.sb[jx] * n0 * n0 + 7.0 / 3.0 * pc.sc[jx] * p73) / n0;
        eps += F * bpow;
        d0 += (dF - 2.0 * jx * F / n0) * bpow;            // d/dn0 at fixed n1: beta^(2j) -> -2j beta^(2j) / n0
        if (jx > 0) d1 += 2.0 * jx * F * bpow / n1;       // d/dn1: 2j beta^(2j) / n1   (n1 = 0: term vanishes with bpow)
        bpow *= b2;
    }
    if (n1 == 0.0) d1 = 0.0;
}

// 1 / g_eff for the spherical cutoff of Eq. 20 (0 where the cutoff momentum is not real: no pairing there)
__device__ __forceinline__ double inv_geff_eq20(double g0r, double M, double U, double mu, double ecut)
{
    const double kc2 = (ecut + mu - U) / M, kf2 = (mu - U) / M;
    if (g0r == 0.0 || !(kc2 > 0.0)) return 0.0;
    const double kc = sqrt(kc2), reg = kc / (4.0 * M_PI * M_PI * M);      // m* k_c / (2 pi^2 hbar^2)
    if (kf2 > 0.0) { const double kf = sqrt(kf2); return 1.0 / g0r - reg * (1.0 - 0.5 * kf / kc * log((kc + kf) / (kc - kf))); }
    const double kp = sqrt(-kf2);
    return 1.0 / g0r - reg * (1.0 + kp / kc * atan(kp / kc));
}

// component i of the vector field of the momentum-coupled external terms at lattice point r:
// Uvec_ext + v_cm + omega x (r - origin)  (Eqs. 24, 26, 36; x_i = i a, Eq. 43)
__device__ __forceinline__ double frame_uvec(const Lattice& L, const PhysConst& pc, const double* uvec, double amp, int i, int r)
{
    const int iz = r % L.nz, iy = (r / L.nz) % L.ny, ix = r / (L.nz * L.ny);
    const double rr[3] = {ix * L.dx - pc.origin[0], iy * L.dx - pc.origin[1], iz * L.dx - pc.origin[2]};
    const int j1 = (i + 1) % 3, j2 = (i + 2) % 3;
    return (uvec ? amp * uvec[(size_t)i * L.nxyz + r] : 0.0) + pc.vcm[i] + pc.omega[j1] * rr[j2] - pc.omega[j2] * rr[j1];
}

__device__ __forceinline__ void load_isopoint(const double* __restrict__ acc_n, const double* __restrict__ acc_p,
                                              const double* __restrict__ gtmp, int nx, int r, IsoPoint& P, double (&kap)[2][2],
                                              double* __restrict__ dens_n, double* __restrict__ dens_p)
{
    const double* acc[2] = {acc_n, acc_p};
    double* dens[2] = {dens_n, dens_p};
    double f[2][19];                                      // species fields in the order of IsoPoint
    for (int q = 0; q < 2; ++q) {
        const double* g = gtmp + (size_t)q * GT_PER_Q * nx;
        const double lap = g[(size_t)GT_LAPN * nx + r];
        f[q][0] = acc[q][(size_t)ACC_N * nx + r];
        f[q][1] = 0.5 * lap - acc[q][(size_t)ACC_T * nx + r];             // tau via Eq. 51
        f[q][2] = lap;
        f[q][3] = g[(size_t)GT_DIVJ * nx + r];
        for (int i = 0; i < 3; ++i) {
            f[q][4 + i] = acc[q][(size_t)(ACC_JC + i) * nx + r];
            f[q][7 + i] = acc[q][(size_t)(ACC_S + i) * nx + r];
            f[q][10 + i] = g[(size_t)(GT_GRADN + i) * nx + r];
            f[q][13 + i] = g[(size_t)(GT_CURLJ + i) * nx + r];
            f[q][16 + i] = g[(size_t)(GT_CURLS + i) * nx + r];
        }
        kap[q][0] = acc[q][(size_t)ACC_K * nx + r]; kap[q][1] = acc[q][(size_t)(ACC_K + 1) * nx + r];
        if (dens[q]) {                                    // Table 2
            double* d = dens[q];
            d[(size_t)D_N * nx + r] = f[q][0]; d[(size_t)D_TAU * nx + r] = f[q][1]; d[(size_t)D_DIVJ * nx + r] = f[q][3];
            d[(size_t)D_KAPPA * nx + r] = kap[q][0]; d[(size_t)(D_KAPPA + 1) * nx + r] = kap[q][1];
            for (int i = 0; i < 3; ++i) {
                d[(size_t)(D_S + i) * nx + r] = f[q][7 + i]; d[(size_t)(D_J + i) * nx + r] = f[q][4 + i];
                d[(size_t)(D_CURLJ + i) * nx + r] = f[q][13 + i];
            }
        }
    }
    for (int t = 0; t < 2; ++t) {
        const double sg = t ? -1.0 : 1.0;
        P.n[t] = f[0][0] + sg * f[1][0]; P.tau[t] = f[0][1] + sg * f[1][1];
        P.lapn[t] = f[0][2] + sg * f[1][2]; P.divJ[t] = f[0][3] + sg * f[1][3];
        for (int i = 0; i < 3; ++i) {
            P.j[t][i] = f[0][4 + i] + sg * f[1][4 + i]; P.s[t][i] = f[0][7 + i] + sg * f[1][7 + i];
            P.gradn[t][i] = f[0][10 + i] + sg * f[1][10 + i]; P.curlj[t][i] = f[0][13 + i] + sg * f[1][13 + i];
            P.curls[t][i] = f[0][16 + i] + sg * f[1][16 + i];
        }
    }
}

// Table-2 densities and the potentials of both species (everything except lap M) from the accumulators.
// Eqs. 13-19 (adopted reading: DESIGN.md section 2), pairing coupling Eqs. 8, 20, 21, Coulomb Eq. 6, external terms
// Eqs. 24, 26, 36.
__global__ void k_potentials(Lattice L, PhysConst pc, ExtFields ext, const double* __restrict__ acc_n, const double* __restrict__ acc_p,
                             const double* __restrict__ gtmp, const double* __restrict__ phi,
                             double* __restrict__ dens_n, double* __restrict__ dens_p,
                             double* __restrict__ pot_n, double* __restrict__ pot_p,
                             double* __restrict__ geff_n, double* __restrict__ geff_p)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    const int nx = L.nxyz;
    if (r >= nx) return;
    IsoPoint P; double kap[2][2];
    load_isopoint(acc_n, acc_p, gtmp, nx, r, P, kap, dens_n, dens_p);
    const double n0 = P.n[0], n1 = P.n[1];
    // ---- isospin fields: U_t = d eps / d n_t, M_t, W_t, S_t, A_t ----
    double U[2], Mt[2], W[2][3], S[2][3], A[2][3];
    const double ng = pow_or_zero(n0, pc.gamma);
    for (int t = 0; t < 2; ++t) {
        U[t] = 2.0 * pc.Cn[t] * P.n[t] + 2.0 * pc.Cg[t] * P.n[t] * ng + 2.0 * pc.Cd[t] * P.lapn[t] + pc.Ct[t] * P.tau[t] + pc.CJ[t] * P.divJ[t];
        Mt[t] = pc.Ct[t] * P.n[t];                                        // d eps / d tau_t
        for (int i = 0; i < 3; ++i) {
            W[t][i] = -pc.CJ[t] * P.gradn[t][i];                          // d eps / d J_t after partial integration (B6)
            S[t][i] = pc.CJ[t] * P.curlj[t][i];                           // d eps / d s_t
            A[t][i] = -pc.Ct[t] * P.j[t][i] + 0.5 * pc.CJ[t] * P.curls[t][i];   // (1/2) d eps / d j_t (B7)
        }
    }
    // n_0^gamma depends on n_0 only: its derivative joins the isoscalar mean field
    U[0] += pc.gamma * pow_or_zero(n0, pc.gamma - 1.0) * (pc.Cg[0] * n0 * n0 + pc.Cg[1] * n1 * n1);
    if (pc.functional == 1) {
        double ev, d0, d1;
        seall1_volume(pc, n0, n1, ev, d0, d1);
        U[0] += d0; U[1] += d1;
    }
    // ---- species basis ----
    double* pot[2] = {pot_n, pot_p};
    double* geff[2] = {geff_n, geff_p};
    double Mq[2], Uq[2], ge[2], g0r[2];
    for (int q = 0; q < 2; ++q) {
        const double xi = q ? -1.0 : 1.0;
        Mq[q] = pc.h2m + Mt[0] + xi * Mt[1];                              // Eq. 13
        Uq[q] = U[0] + xi * U[1];
        g0r[q] = pc.g0[q] * (1.0 - pc.alpha * n0 / 0.16);                 // Eq. 8
        ge[q] = (g0r[q] != 0.0 && pc.cutoff == 0) ? 1.0 / (1.0 / g0r[q] - pc.Kc / (8.0 * M_PI * pc.a * Mq[q])) : 0.0;   // Eq. 21
    }
    if (pc.coulomb) {                                                     // Eq. 6: direct + Slater exchange, protons
        const double np_ = 0.5 * (n0 - n1);
        Uq[1] += phi[r] - pc.e2 * cbrt(3.0 / M_PI) * cbrt(np_ > 0.0 ? np_ : 0.0);
    }
    if (pc.cutoff == 1) {                                                 // Eq. 20 (no rearrangement term: reading B30)
        for (int q = 0; q < 2; ++q) {
            const double inv = inv_geff_eq20(g0r[q], Mq[q], Uq[q], pc.mu[q], pc.ecut);
            ge[q] = inv != 0.0 ? 1.0 / inv : 0.0;
        }
    } else if (pc.rearr) {
        // E_pair = sum_q' g_eff,q' |kappa_q'|^2 depends on the densities through m*_q' (Eq. 21) and g0(n) (Eq. 8):
        // d g_eff = g_eff^2 [ d g0(n) / g0(n)^2 - K dM / (8 pi a M^2) ],  dM_q'/dn_q = Ct0 + xi_q xi_q' Ct1
        double r0 = 0.0, r1 = 0.0;                                        // isoscalar / isovector parts of dE_pair/dn
        for (int qp = 0; qp < 2; ++qp) {
            if (ge[qp] == 0.0) continue;
            const double w = (kap[qp][0] * kap[qp][0] + kap[qp][1] * kap[qp][1]) * ge[qp] * ge[qp];
            const double dm = -w * pc.Kc / (8.0 * M_PI * pc.a * Mq[qp] * Mq[qp]);
            r0 += dm * pc.Ct[0] - w * pc.g0[qp] * pc.alpha / (0.16 * g0r[qp] * g0r[qp]);
            r1 += dm * (qp ? -1.0 : 1.0) * pc.Ct[1];
        }
        Uq[0] += r0 + r1; Uq[1] += r0 - r1;
    }
    for (int q = 0; q < 2; ++q) {
        const double xi = q ? -1.0 : 1.0;
        double* p = pot[q];
        geff[q][r] = ge[q];
        p[(size_t)P_U * nx + r] = Uq[q] + (ext.u0[q] ? ext.amp * ext.u0[q][r] : 0.0);
        p[(size_t)P_M * nx + r] = Mq[q];
        for (int i = 0; i < 3; ++i) {
            p[(size_t)(P_W + i) * nx + r] = W[0][i] + xi * W[1][i];                               // Eq. 16
            p[(size_t)(P_S + i) * nx + r] = S[0][i] + xi * S[1][i] - 0.5 * pc.hbarc * pc.omega[i];   // Eq. 17, - omega . s (Eq. 36)
            // Eq. 18; -(1/2)[Uvec . p + p . Uvec] = -i [A . D + D . A] with A = -(hbar c / 2) Uvec (Eqs. 24, 26, 36)
            p[(size_t)(P_A + i) * nx + r] = A[0][i] + xi * A[1][i] - 0.5 * pc.hbarc * frame_uvec(L, pc, ext.uvec[q], ext.amp, i, r);
        }
        p[(size_t)P_DELTA * nx + r] = -ge[q] * kap[q][0];                                         // Eq. 19
        p[(size_t)(P_DELTA + 1) * nx + r] = -ge[q] * kap[q][1];
    }
}

// row 14: U + lap(M)/2 (the local potential the H-apply kernels read)
__global__ void k_uloc(int nx, double* __restrict__ pot_n, double* __restrict__ pot_p)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nx) return;
    pot_n[(size_t)P_ULOC * nx + r] = pot_n[(size_t)P_U * nx + r] + 0.5 * pot_n[(size_t)P_LAPM * nx + r];
    pot_p[(size_t)P_ULOC * nx + r] = pot_p[(size_t)P_U * nx + r] + 0.5 * pot_p[(size_t)P_LAPM * nx + r];
}

// block-wide sums of NV per-thread values -> out[block][NV] (fixed order: deterministic)
template <int NV>
__device__ __forceinline__ void block_sums(double (&v)[NV], double* __restrict__ out, double scale)
{
    __shared__ double s_red[NV][32];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double x = v[k];
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if (l == 0) s_red[k][w] = x;
    }
    __syncthreads();
    if (threadIdx.x < NV) {
        double t = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += s_red[threadIdx.x][i];
        out[blockIdx.x * NV + threadIdx.x] = t * scale;
    }
}

// energy (Eqs. 4-10): out[block][0..3] = kinetic, functional, Coulomb, pairing; [4..5] = N_n, N_p
__global__ void k_energy(Lattice L, PhysConst pc, const double* __restrict__ acc_n, const double* __restrict__ acc_p,
                         const double* __restrict__ gtmp, const double* __restrict__ phi,
                         const double* __restrict__ geff_n, const double* __restrict__ geff_p, double* __restrict__ out)
{
    const int nx = L.nxyz;
    double e[6] = {0, 0, 0, 0, 0, 0};
    const double* ge[2] = {geff_n, geff_p};
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < nx; r += gridDim.x * blockDim.x) {
        IsoPoint P; double kap[2][2];
        load_isopoint(acc_n, acc_p, gtmp, nx, r, P, kap, nullptr, nullptr);
        const double ng = pow_or_zero(P.n[0], pc.gamma);
        e[0] += pc.h2m * P.tau[0];                                                                 // Eq. 5, bare mass (B9)
        for (int t = 0; t < 2; ++t) {
            double jj = 0.0, sc = 0.0;
            for (int i = 0; i < 3; ++i) { jj += P.j[t][i] * P.j[t][i]; sc += P.s[t][i] * P.curlj[t][i]; }
            e[1] += P.n[t] * (pc.Cn[t] * P.n[t] + pc.Cg[t] * P.n[t] * ng + pc.Cd[t] * P.lapn[t] + pc.Ct[t] * P.tau[t] + pc.CJ[t] * P.divJ[t])
                  - pc.Ct[t] * jj + pc.CJ[t] * sc;                                                 // Eq. 9
        }
        if (pc.functional == 1) { double ev, d0, d1; seall1_volume(pc, P.n[0], P.n[1], ev, d0, d1); e[1] += ev; }
        for (int q = 0; q < 2; ++q) e[3] += ge[q][r] * (kap[q][0] * kap[q][0] + kap[q][1] * kap[q][1]);   // Eq. 7
        const double nn = 0.5 * (P.n[0] + P.n[1]), np_ = 0.5 * (P.n[0] - P.n[1]);
        if (pc.coulomb) e[2] += 0.5 * np_ * phi[r] - 0.75 * pc.e2 * cbrt(3.0 / M_PI) * pow_or_zero(np_, 4.0 / 3.0);   // Eq. 6
        e[4] += nn; e[5] += np_;
    }
    block_sums<6>(e, out, L.dV);
}

// ------------------------------------------------------------------------------------------------
// Observables of PAPER.md Eqs. 37-41 as grid reductions of the Table-2 / Table-3 fields (coordinates x_i = i a).
// pass 1: out[block][16] = N_n, N_p, sum r n_n (3), sum r n_p (3), sum j (3), sum |Delta_n| n_n, sum |Delta_p| n_p,
//         sum_q j_q^2 / n_q, external-term energy density, (unused)
// pass 2 (needs the total centre of mass): out[block][8] = Q20, Q30, Q40, Re Q21, Im Q21, Re Q22, Im Q22, (unused)
// ------------------------------------------------------------------------------------------------
__global__ void k_moments1(Lattice L, PhysConst pc, ExtFields ext, const double* __restrict__ dens_n, const double* __restrict__ dens_p,
                           const double* __restrict__ pot_n, const double* __restrict__ pot_p, double* __restrict__ out)
{
    const int nx = L.nxyz;
    double v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = 0.0;
    const double* d[2] = {dens_n, dens_p};
    const double* p[2] = {pot_n, pot_p};
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < nx; r += gridDim.x * blockDim.x) {
        const int iz = r % L.nz, iy = (r / L.nz) % L.ny, ix = r / (L.nz * L.ny);
        const double x[3] = {ix * L.dx, iy * L.dx, iz * L.dx};
        for (int q = 0; q < 2; ++q) {
            const double n = d[q][(size_t)D_N * nx + r];
            v[q] += n;
            double j2 = 0.0;
            for (int i = 0; i < 3; ++i) {
                const double ji = d[q][(size_t)(D_J + i) * nx + r];
                v[2 + 3 * q + i] += x[i] * n;
                v[8 + i] += ji;
                j2 += ji * ji;
                v[14] += -pc.hbarc * frame_uvec(L, pc, ext.uvec[q], ext.amp, i, r) * ji - 0.5 * pc.hbarc * pc.omega[i] * d[q][(size_t)(D_S + i) * nx + r];
            }
            v[11 + q] += hypot(p[q][(size_t)P_DELTA * nx + r], p[q][(size_t)(P_DELTA + 1) * nx + r]) * n;   // Eq. 39
            if (n > 0.0) v[13] += pc.h2m * j2 / n;                                                        // Eq. 40 (B31)
            if (ext.u0[q]) v[14] += ext.amp * ext.u0[q][r] * n;
        }
    }
    block_sums<16>(v, out, L.dV);
}
__global__ void k_moments2(Lattice L, const double* __restrict__ dens_n, const double* __restrict__ dens_p,
                           double cx, double cy, double cz, double* __restrict__ out)
{
    const int nx = L.nxyz;
    double v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = 0.0;
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < nx; r += gridDim.x * blockDim.x) {
        const int iz = r % L.nz, iy = (r / L.nz) % L.ny, ix = r / (L.nz * L.ny);
        const double x = ix * L.dx - cx, y = iy * L.dx - cy, z = iz * L.dx - cz, r2 = x * x + y * y + z * z;
        const double n = dens_n[r] + dens_p[r];
        v[0] += (2.0 * z * z - x * x - y * y) * n;                         // Eq. 38b
        v[1] += z * (2.0 * z * z - 3.0 * x * x - 3.0 * y * y) * n;         // Eq. 38c
        v[2] += (35.0 * z * z * z * z - 30.0 * z * z * r2 + 3.0 * r2 * r2) * n;   // Eq. 38d
        v[3] += x * z * n; v[4] += y * z * n;                              // Eq. 38e: (x + iy) z
        v[5] += (x * x - y * y) * n; v[6] += 2.0 * x * y * n;              //          (x + iy)^2
    }
    block_sums<8>(v, out, L.dV);
}

// (f)4 boost, Eq. 23: u -> e^{i chi} u, v -> e^{-i chi} v.   grid (blocks over Nxyz, 4 components, states)
__global__ void k_boost(cplx* __restrict__ psi, const double* __restrict__ chi, int nx)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nx) return;
    double sn, cs;
    sincos(chi[r], &sn, &cs);
    if (blockIdx.y >= 2) sn = -sn;
    cplx* p = psi + ((size_t)blockIdx.z * 4 + blockIdx.y) * nx + r;
    const cplx v = *p;
    *p = cmk(v.x * cs - v.y * sn, v.x * sn + v.y * cs);
}
// (f)2 renormalisation, L637: psi_k <- psi_k / sqrt(<psi_k|psi_k>).  nrm[k] = dV sum |psi_k|^2 first (one block per state)
__global__ void k_state_norms(const cplx* __restrict__ psi, size_t slen, double dV, double* __restrict__ nrm)
{
    __shared__ double s_red[32];
    const cplx* a = psi + (size_t)blockIdx.x * slen;
    double s = 0.0;
    for (size_t i = threadIdx.x; i < slen; i += blockDim.x) { const cplx v = a[i]; s = fma(v.x, v.x, fma(v.y, v.y, s)); }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += s_red[i];
        nrm[blockIdx.x] = t * dV;
    }
}
__global__ void k_state_scale(cplx* __restrict__ psi, size_t slen, const double* __restrict__ nrm)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= slen) return;
    const double f = rsqrt(nrm[blockIdx.y]);
    cplx* p = psi + (size_t)blockIdx.y * slen + i;
    const cplx v = *p;
    *p = cmk(v.x * f, v.y * f);
}

// ------------------------------------------------------------------------------------------------
// Coulomb: PAPER.md Eqs. 58-62 evaluated directly on the zero-padded cube of side P = 3 max(N):
//   Phi = (e^2 / P^3) sum_k n~(k) f~(k) e^{ik.r},  f~ = 4 pi (1 - cos kD)/k^2, f~(0) = 2 pi D^2,
//   D = sqrt(3) a max(N).  The DFT passes skip the padded zeros on input and the outputs outside the
//   box ("pruned" transforms), which makes dense passes cheaper than the 27-shift split of Eq. 68.
// out[o][k][i] = sum_{m < nin} in[o][m][i] w^{sgn k m},  w = e^{-2 pi i / P} (tw[r] = w^r)
// ------------------------------------------------------------------------------------------------
__global__ void k_dft_pass_real(const double* __restrict__ in, cplx* __restrict__ out, const cplx* __restrict__ tw,
                                int outer, int nin, int nout, int inner, int P)
{
    const size_t tot = (size_t)outer * nout * inner;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= tot) return;
    const int i = (int)(t % inner); const int k = (int)((t / inner) % nout); const size_t o = t / ((size_t)inner * nout);
    const double* src = in + o * (size_t)nin * inner + i;
    double sr = 0.0, si = 0.0; int idx = 0;
    for (int m = 0; m < nin; ++m) {
        const cplx w = tw[idx]; const double x = src[(size_t)m * inner];
        sr = fma(x, w.x, sr); si = fma(x, w.y, si);
        idx += k; if (idx >= P) idx -= P;
    }
    out[t] = cmk(sr, si);
}
template <int SGN>   // +1 forward (w^{km}), -1 inverse (conj)
__global__ void k_dft_pass(const cplx* __restrict__ in, cplx* __restrict__ out, const cplx* __restrict__ tw,
                           int outer, int nin, int nout, int inner, int P)
{
    const size_t tot = (size_t)outer * nout * inner;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= tot) return;
    const int i = (int)(t % inner); const int k = (int)((t / inner) % nout); const size_t o = t / ((size_t)inner * nout);
    const cplx* src = in + o * (size_t)nin * inner + i;
    double sr = 0.0, si = 0.0; int idx = 0;
    for (int m = 0; m < nin; ++m) {
        cplx w = tw[idx]; if (SGN < 0) w.y = -w.y;
        const cplx x = src[(size_t)m * inner];
        sr = fma(x.x, w.x, sr); sr = fma(-x.y, w.y, sr);
        si = fma(x.x, w.y, si); si = fma(x.y, w.x, si);
        idx += k; if (idx >= P) idx -= P;
    }
    out[t] = cmk(sr, si);
}
__global__ void k_coulomb_kernel_mult(cplx* __restrict__ A, int P, double a, double Dc)
{
    const size_t tot = (size_t)P * P * P;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= tot) return;
    const int kz = (int)(t % P), ky = (int)((t / P) % P), kx = (int)(t / ((size_t)P * P));
    const double c = 2.0 * M_PI / (P * a);
    const double qx = c * (2 * kx < P ? kx : kx - P), qy = c * (2 * ky < P ? ky : ky - P), qz = c * (2 * kz < P ? kz : kz - P);
    const double k2 = qx * qx + qy * qy + qz * qz;
    const double ft = (k2 == 0.0) ? 2.0 * M_PI * Dc * Dc : 4.0 * M_PI * (1.0 - cos(sqrt(k2) * Dc)) / k2;
    cplx v = A[t];
    A[t] = cmk(v.x * ft, v.y * ft);
}
__global__ void k_dft_pass_final(const cplx* __restrict__ in, double* __restrict__ out, const cplx* __restrict__ tw,
                                 int outer, int nin, int nout, int P, double scale)
{
    const size_t tot = (size_t)outer * nout;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= tot) return;
    const int k = (int)(t % nout); const size_t o = t / nout;
    const cplx* src = in + o * (size_t)nin;
    double sr = 0.0; int idx = 0;
    for (int m = 0; m < nin; ++m) {
        const cplx w = tw[idx]; const cplx x = src[m];
        sr = fma(x.x, w.x, sr); sr = fma(x.y, w.y, sr);     // Re( x conj(w) )
        idx += k; if (idx >= P) idx -= P;
    }
    out[t] = scale * sr;
}
