// grid_kernels.cuh -- grid-only work between the two global barriers of a time step:
// density reduction, lattice derivatives of real fields, Skyrme/pairing potentials, Coulomb, energy.
// All fields are Nxyz doubles; the work is tiny next to the per-state kernels, so these kernels are
// written for clarity and launch count, not for peak throughput.
#pragma once
#include "common.cuh"

struct PhysConst {
    double h2m, e2, hbarc, gamma, a, Kc;
    double Cn[2], Cg[2], Cd[2], Ct[2], CJ[2], g0[2];
    int coulomb, rearr;
};

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

__device__ __forceinline__ double powpos(double x, double p) { return x > 0.0 ? pow(x, p) : 0.0; }

// Table-2 densities, potentials of both species (everything except lap M), g_eff.   Adopted reading:
// DESIGN.md / SURVEY.md Appendix A.3 (Eqs. 13-19, 21, 6).
__global__ void k_potentials(Lattice L, PhysConst pc, const double* __restrict__ acc_n, const double* __restrict__ acc_p,
                             const double* __restrict__ gtmp, const double* __restrict__ phi,
                             double* __restrict__ dens_n, double* __restrict__ dens_p,
                             double* __restrict__ pot_n, double* __restrict__ pot_p,
                             double* __restrict__ geff_n, double* __restrict__ geff_p)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    const int nx = L.nxyz;
    if (r >= nx) return;
    const double* acc[2] = {acc_n, acc_p};
    double* dens[2] = {dens_n, dens_p};
    double* pot[2] = {pot_n, pot_p};
    double* geff[2] = {geff_n, geff_p};
    double n[2], tau[2], lapn[2], divJ[2], kr[2], ki[2];
    double s[2][3], j[2][3], gradn[2][3], curlj[2][3], curls[2][3];
    for (int q = 0; q < 2; ++q) {
        const double* g = gtmp + (size_t)q * GT_PER_Q * nx;
        n[q] = acc[q][(size_t)ACC_N * nx + r];
        lapn[q] = g[(size_t)GT_LAPN * nx + r];
        tau[q] = 0.5 * lapn[q] - acc[q][(size_t)ACC_T * nx + r];          // Eq. 51
        divJ[q] = g[(size_t)GT_DIVJ * nx + r];
        kr[q] = acc[q][(size_t)ACC_K * nx + r]; ki[q] = acc[q][(size_t)(ACC_K + 1) * nx + r];
        for (int i = 0; i < 3; ++i) {
            s[q][i] = acc[q][(size_t)(ACC_S + i) * nx + r];
            j[q][i] = acc[q][(size_t)(ACC_JC + i) * nx + r];
            gradn[q][i] = g[(size_t)(GT_GRADN + i) * nx + r];
            curlj[q][i] = g[(size_t)(GT_CURLJ + i) * nx + r];
            curls[q][i] = g[(size_t)(GT_CURLS + i) * nx + r];
        }
        // Table 2
        double* d = dens[q];
        d[(size_t)D_N * nx + r] = n[q]; d[(size_t)D_TAU * nx + r] = tau[q]; d[(size_t)D_DIVJ * nx + r] = divJ[q];
        d[(size_t)D_KAPPA * nx + r] = kr[q]; d[(size_t)(D_KAPPA + 1) * nx + r] = ki[q];
        for (int i = 0; i < 3; ++i) {
            d[(size_t)(D_S + i) * nx + r] = s[q][i]; d[(size_t)(D_J + i) * nx + r] = j[q][i];
            d[(size_t)(D_CURLJ + i) * nx + r] = curlj[q][i];
        }
    }
    const double n0 = n[0] + n[1], n1 = n[0] - n[1];
    const double xi[2] = {1.0, -1.0};
    double M[2], ge[2];
    for (int q = 0; q < 2; ++q) {
        M[q] = pc.h2m + pc.Ct[0] * n0 + xi[q] * pc.Ct[1] * n1;                                    // Eq. 13
        ge[q] = (pc.g0[q] != 0.0) ? 1.0 / (1.0 / pc.g0[q] - pc.Kc / (8.0 * M_PI * pc.a * M[q])) : 0.0;   // Eq. 21
        geff[q][r] = ge[q];
    }
    const double pg1 = powpos(n0, pc.gamma + 1.0), pg0 = powpos(n0, pc.gamma), pgm = powpos(n0, pc.gamma - 1.0);
    for (int q = 0; q < 2; ++q) {
        const double x = xi[q];
        double u = 2.0 * pc.Cn[0] * n0 + 2.0 * x * pc.Cn[1] * n1
                 + pc.Ct[0] * (tau[0] + tau[1]) + x * pc.Ct[1] * (tau[0] - tau[1])
                 + 2.0 * pc.Cd[0] * (lapn[0] + lapn[1]) + 2.0 * x * pc.Cd[1] * (lapn[0] - lapn[1])
                 + pc.CJ[0] * (divJ[0] + divJ[1]) + x * pc.CJ[1] * (divJ[0] - divJ[1])
                 + (pc.gamma + 2.0) * pc.Cg[0] * pg1 + 2.0 * x * pc.Cg[1] * n1 * pg0
                 + pc.gamma * pc.Cg[1] * n1 * n1 * pgm;
        if (pc.rearr)
            for (int qp = 0; qp < 2; ++qp) {
                if (pc.g0[qp] == 0.0) continue;
                const double k2 = kr[qp] * kr[qp] + ki[qp] * ki[qp];
                const double dg = -ge[qp] * ge[qp] * pc.Kc / (8.0 * M_PI * pc.a * M[qp] * M[qp]);
                u += k2 * dg * (pc.Ct[0] + x * xi[qp] * pc.Ct[1]);
            }
        if (q == 1 && pc.coulomb) {
            const double npr = n[1] > 0.0 ? n[1] : 0.0;
            u += phi[r] - pc.e2 * cbrt(3.0 / M_PI) * cbrt(npr);                                   // Eq. 6
        }
        double* p = pot[q];
        p[(size_t)P_U * nx + r] = u;
        p[(size_t)P_M * nx + r] = M[q];
        for (int i = 0; i < 3; ++i) {
            p[(size_t)(P_W + i) * nx + r] = -(pc.CJ[0] * (gradn[0][i] + gradn[1][i]) + x * pc.CJ[1] * (gradn[0][i] - gradn[1][i]));
            p[(size_t)(P_S + i) * nx + r] = pc.CJ[0] * (curlj[0][i] + curlj[1][i]) + x * pc.CJ[1] * (curlj[0][i] - curlj[1][i]);
            p[(size_t)(P_A + i) * nx + r] = -(pc.Ct[0] * (j[0][i] + j[1][i]) + x * pc.Ct[1] * (j[0][i] - j[1][i]))
                                          + 0.5 * (pc.CJ[0] * (curls[0][i] + curls[1][i]) + x * pc.CJ[1] * (curls[0][i] - curls[1][i]));
        }
        p[(size_t)P_DELTA * nx + r] = -ge[q] * kr[q];                                             // Eq. 19
        p[(size_t)(P_DELTA + 1) * nx + r] = -ge[q] * ki[q];
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

// energy density of SURVEY.md A.8 (Eqs. 4-9): out[block][0..3] = kin, skyrme, coul, pair; [4..5] = N_n, N_p
__global__ void k_energy(Lattice L, PhysConst pc, const double* __restrict__ dens_n, const double* __restrict__ dens_p,
                         const double* __restrict__ gtmp, const double* __restrict__ phi,
                         const double* __restrict__ geff_n, const double* __restrict__ geff_p, double* __restrict__ out)
{
    __shared__ double s_red[6][32];
    const int nx = L.nxyz;
    double e[6] = {0, 0, 0, 0, 0, 0};
    const double* d[2] = {dens_n, dens_p};
    const double* ge[2] = {geff_n, geff_p};
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < nx; r += gridDim.x * blockDim.x) {
        double nq[2] = {d[0][r], d[1][r]};
        const double n0 = nq[0] + nq[1];
        e[0] += pc.h2m * (d[0][(size_t)D_TAU * nx + r] + d[1][(size_t)D_TAU * nx + r]);
        for (int t = 0; t < 2; ++t) {
            const double sg = t ? -1.0 : 1.0;
            const double nt = nq[0] + sg * nq[1];
            const double taut = d[0][(size_t)D_TAU * nx + r] + sg * d[1][(size_t)D_TAU * nx + r];
            const double lapt = gtmp[(size_t)GT_LAPN * nx + r] + sg * gtmp[(size_t)(GT_PER_Q + GT_LAPN) * nx + r];
            const double divt = d[0][(size_t)D_DIVJ * nx + r] + sg * d[1][(size_t)D_DIVJ * nx + r];
            double jj = 0.0, scj = 0.0;
            for (int i = 0; i < 3; ++i) {
                const double jt = d[0][(size_t)(D_J + i) * nx + r] + sg * d[1][(size_t)(D_J + i) * nx + r];
                const double st = d[0][(size_t)(D_S + i) * nx + r] + sg * d[1][(size_t)(D_S + i) * nx + r];
                const double ct = d[0][(size_t)(D_CURLJ + i) * nx + r] + sg * d[1][(size_t)(D_CURLJ + i) * nx + r];
                jj += jt * jt; scj += st * ct;
            }
            e[1] += pc.Cn[t] * nt * nt + pc.Cg[t] * nt * nt * powpos(n0, pc.gamma) + pc.Cd[t] * nt * lapt
                  + pc.Ct[t] * (nt * taut - jj) + pc.CJ[t] * (nt * divt + scj);
        }
        for (int q = 0; q < 2; ++q) {
            const double kr = d[q][(size_t)D_KAPPA * nx + r], ki = d[q][(size_t)(D_KAPPA + 1) * nx + r];
            e[3] += ge[q][r] * (kr * kr + ki * ki);
        }
        if (pc.coulomb) {
            const double npr = nq[1] > 0.0 ? nq[1] : 0.0;
            e[2] += 0.5 * nq[1] * phi[r] - 0.75 * pc.e2 * cbrt(3.0 / M_PI) * pow(npr, 4.0 / 3.0);
        }
        e[4] += nq[0]; e[5] += nq[1];
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    for (int k = 0; k < 6; ++k) {
        double v = e[k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (l == 0) s_red[k][w] = v;
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double t = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += s_red[threadIdx.x][i];
        out[blockIdx.x * 6 + threadIdx.x] = t * L.dV;
    }
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
