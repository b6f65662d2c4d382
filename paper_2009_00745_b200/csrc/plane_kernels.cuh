// plane_kernels.cuh -- the per-state kernels on the fp64 tensor-core path ("v3").
//
// Same decomposition as state_kernels.cuh (h = V_loc + sum_i T_i, T_i acting on lattice lines, a CTA works
// on one lattice plane in shared memory), re-organised around the DMMA line operator:
//   * a CTA OWNS one plane for the whole launch and loops over states (grid = planes x G groups, sized to
//     the SM count): the potentials of the plane (M, B_i = A_i + (sigma x W)_i / 2) are staged in shared
//     memory once, the density accumulators of the plane stay in shared memory across the state loop;
//   * one fused pass per in-plane axis: a warp task = one 2-spinor x one strip of 4 lines.  Per k step it
//     loads phi_up, phi_dn and the potentials at 4 points of each line, forms g = C phi (C = -i B) and
//     q = -M phi / 2 in registers, and feeds the tiles  a += c1 phi, b += c2 phi, acc += c1 g + c2 q
//     (c1, c2: circulant tiles of D_i, D2_i, Eq. 48).  The epilogue applies
//     T_i phi = C a - M b / 2 + acc at the thread's own output point: no intermediate array, no extra sync.
// MMA tile mapping (m8n8k4, thread g = lane / 4, t = lane % 4):  out[n][col] = sum_m c[n - m] x[m][col],
//   A = circulant tile (row 8r+g, k 4k+t), B = x tile (k 4k+t, column g = (line l0 + g/2, re|im)),
//   accumulator row 8r+g, columns 2t, 2t+1 = (re, im) of line l0 + t.  Lines are addressed by
//   (line stride LS, point stride PS), so the two in-plane axes run the same code.
// Requires every lattice edge to be a multiple of 4 (rows padded to a multiple of 8 inside the tiles).
#pragma once
#include "common.cuh"
#include "state_kernels.cuh"

template <int N>
struct LineT {
    static constexpr int NK = N / 4;                           // k steps
    static constexpr int NT = (N + 7) / 8;                     // output row tiles
    static constexpr int RT = (NT <= 5) ? NT : (NT + 1) / 2;   // row tiles per pass (bounds the accumulators)
};

__device__ __forceinline__ void dmma2(double (&d)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

// circulant fragments of this thread: cf[j] = c[(4j + g - t) mod N]   (ct: doubled table, ct[N + d])
template <int N>
__device__ __forceinline__ void load_cf(const double2* __restrict__ ct, int g, int t, double (&cf1)[N / 4], double (&cf2)[N / 4])
{
#pragma unroll
    for (int j = 0; j < N / 4; ++j) {
        const int d = (4 * j + g - t + N) % N;
        const double2 c = ct[N + d];
        cf1[j] = c.x; cf2[j] = c.y;
    }
}

// potentials of one plane for one axis, in shared memory
struct AxisPot {
    const double* M;      // hbar^2 / 2m*
    const double2* D;     // (B00, B11)
    const double2* O;     // B01 (re, im)
};

// T_i phi of one 2-spinor on a strip of 4 lines, accumulated into out_u / out_d.
template <int N>
__device__ __forceinline__ void happly_axis_task(const cplx* __restrict__ phi_u, const cplx* __restrict__ phi_d,
                                                 cplx* __restrict__ out_u, cplx* __restrict__ out_d,
                                                 const AxisPot pot, int l0, int LS, int PS, const double2* __restrict__ ct)
{
    typedef LineT<N> T;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    double cf1[T::NK], cf2[T::NK];
    load_cf<N>(ct, g, t, cf1, cf2);
    const bool im = g & 1;
    const int ibase = (l0 + (g >> 1)) * LS + t * PS;
    const int obase = (l0 + t) * LS + g * PS;
#pragma unroll
    for (int r0 = 0; r0 < T::NT; r0 += T::RT) {
        double au[T::RT][2], ad[T::RT][2], bu[T::RT][2], bd[T::RT][2], cu[T::RT][2], cd[T::RT][2];
#pragma unroll
        for (int r = 0; r < T::RT; ++r) {
            au[r][0] = au[r][1] = ad[r][0] = ad[r][1] = 0.0;
            bu[r][0] = bu[r][1] = bd[r][0] = bd[r][1] = 0.0;
            cu[r][0] = cu[r][1] = cd[r][0] = cd[r][1] = 0.0;
        }
#pragma unroll
        for (int k = 0; k < T::NK; ++k) {
            const int ii = ibase + 4 * k * PS;
            const cplx fu = phi_u[ii], fd = phi_d[ii];
            const double M = pot.M[ii];
            const double2 D = pot.D[ii], O = pot.O[ii];
            cplx gu, gd;
            apply_C(D.x, D.y, cmk(O.x, O.y), fu, fd, gu, gd);                 // g = C phi
            const double xfu = im ? fu.y : fu.x, xfd = im ? fd.y : fd.x;
            const double xgu = im ? gu.y : gu.x, xgd = im ? gd.y : gd.x;
            const double xqu = -0.5 * M * xfu, xqd = -0.5 * M * xfd;          // q = -M phi / 2
#pragma unroll
            for (int r = 0; r < T::RT; ++r) {
                if (r0 + r >= T::NT) continue;
                const int j = (((2 * (r0 + r) - k) % T::NK) + T::NK) % T::NK;
                dmma2(au[r], cf1[j], xfu); dmma2(ad[r], cf1[j], xfd);
                dmma2(bu[r], cf2[j], xfu); dmma2(bd[r], cf2[j], xfd);
                dmma2(cu[r], cf1[j], xgu); dmma2(cd[r], cf1[j], xgd);
                dmma2(cu[r], cf2[j], xqu); dmma2(cd[r], cf2[j], xqd);
            }
        }
#pragma unroll
        for (int r = 0; r < T::RT; ++r) {
            if (r0 + r >= T::NT) continue;
            if (8 * (r0 + r) + g >= N) continue;                              // padding rows
            const int oi = obase + 8 * (r0 + r) * PS;
            const double M = pot.M[oi];
            const double2 D = pot.D[oi], O = pot.O[oi];
            cplx lu, ld_;
            apply_C(D.x, D.y, cmk(O.x, O.y), cmk(au[r][0], au[r][1]), cmk(ad[r][0], ad[r][1]), lu, ld_);   // C D phi
            const cplx ou = out_u[oi], od = out_d[oi];
            out_u[oi] = cmk(ou.x + lu.x - 0.5 * M * bu[r][0] + cu[r][0], ou.y + lu.y - 0.5 * M * bu[r][1] + cu[r][1]);
            out_d[oi] = cmk(od.x + ld_.x - 0.5 * M * bd[r][0] + cd[r][0], od.y + ld_.y - 0.5 * M * bd[r][1] + cd[r][1]);
        }
    }
}

// density contributions of one axis (Eq. 3 with phi = conj(v), tau via Eq. 51) on a strip of 4 lines,
// accumulated into the shared-memory planes dens[f * P + point].  WHICH = 0: first-derivative terms
// (j_axis, J), 1: second-derivative term (t); the two halves are separate warp tasks (load balance).
template <int N, int WHICH>
__device__ __forceinline__ void dens_axis_task(const cplx* __restrict__ phi_u, const cplx* __restrict__ phi_d,
                                               double* __restrict__ dens, int P, int axis,
                                               int l0, int LS, int PS, const double2* __restrict__ ct)
{
    typedef LineT<N> T;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    double cf1[T::NK], cf2[T::NK];
    load_cf<N>(ct, g, t, cf1, cf2);
    const bool im = g & 1;
    const int ibase = (l0 + (g >> 1)) * LS + t * PS;
    const int obase = (l0 + t) * LS + g * PS;
#pragma unroll
    for (int r0 = 0; r0 < T::NT; r0 += T::RT) {
        double au[T::RT][2], ad[T::RT][2];
#pragma unroll
        for (int r = 0; r < T::RT; ++r) au[r][0] = au[r][1] = ad[r][0] = ad[r][1] = 0.0;
#pragma unroll
        for (int k = 0; k < T::NK; ++k) {
            const int ii = ibase + 4 * k * PS;
            const cplx fu = phi_u[ii], fd = phi_d[ii];
            const double xfu = im ? fu.y : fu.x, xfd = im ? fd.y : fd.x;
#pragma unroll
            for (int r = 0; r < T::RT; ++r) {
                if (r0 + r >= T::NT) continue;
                const int j = (((2 * (r0 + r) - k) % T::NK) + T::NK) % T::NK;
                const double c = (WHICH == 0) ? cf1[j] : cf2[j];
                dmma2(au[r], c, xfu); dmma2(ad[r], c, xfd);
            }
        }
#pragma unroll
        for (int r = 0; r < T::RT; ++r) {
            if (r0 + r >= T::NT) continue;
            if (8 * (r0 + r) + g >= N) continue;
            const int oi = obase + 8 * (r0 + r) * PS;
            const cplx fu = phi_u[oi], fd = phi_d[oi];
            const cplx du = cmk(au[r][0], au[r][1]), dd = cmk(ad[r][0], ad[r][1]);
            if (WHICH == 1) {
                dens[ACC_T * P + oi] += fu.x * du.x + fu.y * du.y + fd.x * dd.x + fd.y * dd.y;
            } else {
                const double ju = fu.x * du.y - fu.y * du.x, jd = fd.x * dd.y - fd.y * dd.x;
                // z1 = conj(phi_up) a_dn, z2 = conj(phi_dn) a_up
                const double z1r = fu.x * dd.x + fu.y * dd.y, z1i = fu.x * dd.y - fu.y * dd.x;
                const double z2r = fd.x * du.x + fd.y * du.y, z2i = fd.x * du.y - fd.y * du.x;
                const double Xx = z1i + z2i, Xy = -z1r + z2r, Xz = ju - jd;
                dens[(ACC_JC + axis) * P + oi] += ju + jd;
                if (axis == 0)      { dens[(ACC_J + 2) * P + oi] += Xy; dens[(ACC_J + 1) * P + oi] -= Xz; }
                else if (axis == 1) { dens[(ACC_J + 0) * P + oi] += Xz; dens[(ACC_J + 2) * P + oi] -= Xx; }
                else                { dens[(ACC_J + 1) * P + oi] += Xx; dens[(ACC_J + 0) * P + oi] -= Xy; }
            }
        }
    }
}

__device__ __forceinline__ void stage_axis_pot(const Lattice& L, const double* __restrict__ pot, int axis, int gi, int si,
                                               double* sM, double2* sD, double2* sO)
{
    const int nxyz = L.nxyz;
    const double A = pot[(size_t)(P_A + axis) * nxyz + gi];
    const double Wx = pot[(size_t)(P_W + 0) * nxyz + gi], Wy = pot[(size_t)(P_W + 1) * nxyz + gi],
                 Wz = pot[(size_t)(P_W + 2) * nxyz + gi];
    double b00, b11; cplx b01;
    make_B(axis, A, Wx, Wy, Wz, b00, b11, b01);
    if (sM) sM[si] = pot[(size_t)P_M * nxyz + gi];
    sD[si] = make_double2(b00, b11);
    sO[si] = b01;
}

// ------------------------------------------------------------------------------------------------
// H-apply, yz-planes:  W = [V_loc + T_y + T_z] X + pairing block.      grid (nx, G), 256 threads
//   NCOMP = 4: both 2-spinors (u pair, conj v pair) of a state in shared memory at once; 2: one after the other
// shared: tables | potM | potD[2] | potO[2] | phi[NCOMP] | out[NCOMP]
// ------------------------------------------------------------------------------------------------
template <int NY, int NZ, int NCOMP>
__global__ void __launch_bounds__(256) k3_happly_yz(HArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int P = NY * NZ;
    const Lattice L = a.L;
    const int nxyz = L.nxyz;
    const int gbase = blockIdx.x * P;
    double2* s_cty = smem;
    double2* s_ctz = s_cty + 2 * NY;
    double2* potD = s_ctz + 2 * NZ;             // [2][P]
    double2* potO = potD + 2 * P;               // [2][P]
    cplx* phi = potO + 2 * P;                   // [NCOMP][P]
    cplx* out = phi + NCOMP * P;                // [NCOMP][P]
    double* potM = (double*)(out + NCOMP * P);  // [P]
    stage_table(s_cty, a.ctab[1], NY);
    stage_table(s_ctz, a.ctab[2], NZ);
    const double* pot = a.pot;
    for (int p = threadIdx.x; p < P; p += blockDim.x) {
        stage_axis_pot(L, pot, 1, gbase + p, p, potM, potD, potO);
        stage_axis_pot(L, pot, 2, gbase + p, p, nullptr, potD + P, potO + P);
    }
    const AxisPot poty = {potM, potD, potO}, potz = {potM, potD + P, potO + P};
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    constexpr int NPAIR = NCOMP / 2;
    __syncthreads();

    for (int st = blockIdx.y; st < a.ns; st += a.G) {
        const cplx* Xs = a.X + (size_t)st * 4 * nxyz;
        cplx* Ws = a.W + (size_t)st * 4 * nxyz;
#pragma unroll 1
        for (int pg = 0; pg < 2 / NPAIR; ++pg) {
            // ---- load the 2-spinors (v pair conjugated) and initialise out = V_loc phi ----
            for (int p = threadIdx.x; p < P; p += blockDim.x) {
                const int gi = gbase + p;
                const double ul = pot[(size_t)P_ULOC * nxyz + gi];
                const double sx = pot[(size_t)(P_S + 0) * nxyz + gi], sy = pot[(size_t)(P_S + 1) * nxyz + gi],
                             sz = pot[(size_t)(P_S + 2) * nxyz + gi];
#pragma unroll
                for (int pr = 0; pr < NPAIR; ++pr) {
                    const int pair = pg * NPAIR + pr;
                    cplx fu = Xs[(size_t)(2 * pair) * nxyz + gi], fd = Xs[(size_t)(2 * pair + 1) * nxyz + gi];
                    if (pair) { fu = cconj(fu); fd = cconj(fd); }
                    phi[(2 * pr) * P + p] = fu; phi[(2 * pr + 1) * P + p] = fd;
                    cplx ou = cscale(ul + sz, fu); cfma(ou, cmk(sx, -sy), fd);
                    cplx od = cscale(ul - sz, fd); cfma(od, cmk(sx, sy), fu);
                    out[(2 * pr) * P + p] = ou; out[(2 * pr + 1) * P + p] = od;
                }
            }
            __syncthreads();
            // ---- y lines (one per z): LS = 1, PS = NZ ----
            for (int task = warp; task < NPAIR * (NZ / 4); task += nwarps) {
                const int pr = task / (NZ / 4), l0 = 4 * (task - pr * (NZ / 4));
                happly_axis_task<NY>(phi + 2 * pr * P, phi + (2 * pr + 1) * P, out + 2 * pr * P, out + (2 * pr + 1) * P,
                                     poty, l0, 1, NZ, s_cty);
            }
            __syncthreads();
            // ---- z lines (one per y): LS = NZ, PS = 1 ----
            for (int task = warp; task < NPAIR * (NY / 4); task += nwarps) {
                const int pr = task / (NY / 4), l0 = 4 * (task - pr * (NY / 4));
                happly_axis_task<NZ>(phi + 2 * pr * P, phi + (2 * pr + 1) * P, out + 2 * pr * P, out + (2 * pr + 1) * P,
                                     potz, l0, NZ, 1, s_ctz);
            }
            __syncthreads();
            // ---- pairing block and write (Eq. 11, mu = 0) ----
            for (int p = threadIdx.x; p < P; p += blockDim.x) {
                const int gi = gbase + p;
                const cplx Dl = cmk(pot[(size_t)P_DELTA * nxyz + gi], pot[(size_t)(P_DELTA + 1) * nxyz + gi]);
#pragma unroll
                for (int pr = 0; pr < NPAIR; ++pr) {
                    const int pair = pg * NPAIR + pr;
                    cplx ou = out[(2 * pr) * P + p], od = out[(2 * pr + 1) * P + p];
                    if (pair == 0) {
                        cplx vu, vd;
                        if (NCOMP == 4) { vu = cconj(phi[2 * P + p]); vd = cconj(phi[3 * P + p]); }
                        else { vu = Xs[(size_t)2 * nxyz + gi]; vd = Xs[(size_t)3 * nxyz + gi]; }
                        cfma(ou, Dl, vd);
                        cfma(od, cmk(-Dl.x, -Dl.y), vu);
                    } else {
                        cplx uu, ud;
                        if (NCOMP == 4) { uu = phi[p]; ud = phi[P + p]; }
                        else { uu = Xs[gi]; ud = Xs[(size_t)nxyz + gi]; }
                        const cplx Dc = cconj(Dl);
                        ou = cmk(-ou.x, ou.y); od = cmk(-od.x, od.y);       // -conj(h conj v)
                        cfma(ou, cmk(-Dc.x, -Dc.y), ud);
                        cfma(od, Dc, uu);
                    }
                    Ws[(size_t)(2 * pair) * nxyz + gi] = ou; Ws[(size_t)(2 * pair + 1) * nxyz + gi] = od;
                }
            }
            __syncthreads();
        }
    }
}

// ------------------------------------------------------------------------------------------------
// H-apply, xz-planes:  W += T_x X,  eta_part[st][iy] = dV Re <X|W> over the plane.   grid (ny, G), 256 threads
// shared: table | potD | potO | phi[NCOMP] | out[NCOMP] | potM | red
// ------------------------------------------------------------------------------------------------
template <int NX, int NCOMP>
__global__ void __launch_bounds__(256) k3_happly_xz(HArgs a)
{
    extern __shared__ double2 smem[];
    const Lattice L = a.L;
    const int nz = L.nz, nxyz = L.nxyz, P = NX * nz, gs = L.ny * nz, gb = blockIdx.x * nz;
    double2* s_ctx = smem;
    double2* potD = s_ctx + 2 * NX;
    double2* potO = potD + P;
    cplx* phi = potO + P;
    cplx* out = phi + NCOMP * P;
    double* potM = (double*)(out + NCOMP * P);
    double* s_red = potM + P;
    stage_table(s_ctx, a.ctab[0], NX);
    for (int p = threadIdx.x; p < P; p += blockDim.x) {
        const int ix = p / nz, iz = p - ix * nz;
        stage_axis_pot(L, a.pot, 0, gb + ix * gs + iz, p, potM, potD, potO);
    }
    const AxisPot potx = {potM, potD, potO};
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    constexpr int NPAIR = NCOMP / 2;
    __syncthreads();

    for (int st = blockIdx.y; st < a.ns; st += a.G) {
        const cplx* Xs = a.X + (size_t)st * 4 * nxyz;
        cplx* Ws = a.W + (size_t)st * 4 * nxyz;
        double eta_loc = 0.0;
#pragma unroll 1
        for (int pg = 0; pg < 2 / NPAIR; ++pg) {
            for (int p = threadIdx.x; p < P; p += blockDim.x) {
                const int ix = p / nz, iz = p - ix * nz, gi = gb + ix * gs + iz;
#pragma unroll
                for (int c = 0; c < NCOMP; ++c) {
                    const int cg = pg * NCOMP + c;
                    cplx f = Xs[(size_t)cg * nxyz + gi];
                    if (cg >= 2) f = cconj(f);
                    phi[c * P + p] = f;
                    out[c * P + p] = cmk(0.0, 0.0);
                }
            }
            __syncthreads();
            // ---- x lines (one per z): LS = 1, PS = nz ----
            for (int task = warp; task < NPAIR * (nz / 4); task += nwarps) {
                const int pr = task / (nz / 4), l0 = 4 * (task - pr * (nz / 4));
                happly_axis_task<NX>(phi + 2 * pr * P, phi + (2 * pr + 1) * P, out + 2 * pr * P, out + (2 * pr + 1) * P,
                                     potx, l0, 1, nz, s_ctx);
            }
            __syncthreads();
            for (int p = threadIdx.x; p < P; p += blockDim.x) {
                const int ix = p / nz, iz = p - ix * nz, gi = gb + ix * gs + iz;
#pragma unroll
                for (int c = 0; c < NCOMP; ++c) {
                    const int cg = pg * NCOMP + c;
                    cplx o = out[c * P + p], x = phi[c * P + p];
                    if (cg >= 2) { o = cmk(-o.x, o.y); x = cconj(x); }
                    cplx* w = Ws + (size_t)cg * nxyz + gi;
                    const cplx tw = cadd(*w, o);
                    *w = tw;
                    eta_loc += x.x * tw.x + x.y * tw.y;
                }
            }
            __syncthreads();
        }
        const double tsum = block_sum(eta_loc, s_red);
        if (threadIdx.x == 0) a.eta_part[(size_t)st * L.ny + blockIdx.x] = tsum * L.dV;
    }
}

// ------------------------------------------------------------------------------------------------
// ABM update fused with the y/z density pass of the NEW state (modes as k_update_yz in state_kernels.cuh).
// grid (nx, G), 256 threads.   shared: tables | phi[2] | dens[13][P] | s_eta
// The plane's density accumulators stay in shared memory over the state loop and are added to
// part[g] once at the end.
// ------------------------------------------------------------------------------------------------
template <int MODE, int NY, int NZ>
__global__ void __launch_bounds__(256) k3_update_yz(UArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int P = NY * NZ;
    const Lattice L = a.L;
    const int nxyz = L.nxyz;
    const int gbase = blockIdx.x * P;
    double2* s_cty = smem;
    double2* s_ctz = s_cty + 2 * NY;
    cplx* phi = s_ctz + 2 * NZ;                       // [2][P]
    double* dens = (double*)(phi + 2 * P);            // [LISE_NACC][P]
    double* s_eta = dens + LISE_NACC * P;
    if (MODE != 3) {
        stage_table(s_cty, a.ctab[1], NY); stage_table(s_ctz, a.ctab[2], NZ);
        for (int i = threadIdx.x; i < LISE_NACC * P; i += blockDim.x) dens[i] = 0.0;
        __syncthreads();
    }
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const double ih = 1.0 / a.hbarc;
    const double c48 = a.dt / 48.0;

    for (int st = blockIdx.y; st < a.ns; st += a.G) {
        const size_t so = (size_t)st * 4 * nxyz;
        double eta = 0.0;
        if (MODE != 0) {
            __syncthreads();
            if (threadIdx.x == 0) {
                double e = 0.0;
                if (MODE == 3 && a.order > 1) e = a.eta_fix[st];
                else {
                    for (int j = 0; j < L.ny; ++j) e += a.eta_part[(size_t)st * L.ny + j];
                    if (!a.remove_phase) e = 0.0;
                    if (MODE == 3 && blockIdx.x == 0) a.eta_fix[st] = e;
                }
                s_eta[0] = e;
            }
            __syncthreads();
            eta = s_eta[0];
        }
        for (int p = threadIdx.x; p < P; p += blockDim.x) {
            const int gi = gbase + p;
            cplx nu0 = cmk(0, 0), nv[2];
            nv[0] = cmk(0, 0); nv[1] = cmk(0, 0);
#pragma unroll
            for (int cp = 0; cp < 4; ++cp) {
                const size_t o = so + (size_t)cp * nxyz + gi;
                cplx nw;
                if (MODE == 0) {
                    nw = a.Z[o];
                } else if (MODE == 1) {
                    const cplx w = a.W[o], y = a.sA[o], ym = a.sB[o], f1 = a.sD[o], f2 = a.sE[o], f3 = a.sC[o], e = a.sF[o];
                    const cplx fn = cmk((w.y - eta * y.y) * ih, -(w.x - eta * y.x) * ih);
                    const cplx half = cmk(0.5 * (y.x + ym.x), 0.5 * (y.y + ym.y));
                    cplx pp, qq;
                    pp.x = half.x + c48 * (119.0 * fn.x - 99.0 * f1.x + 69.0 * f2.x - 17.0 * f3.x);
                    pp.y = half.y + c48 * (119.0 * fn.y - 99.0 * f1.y + 69.0 * f2.y - 17.0 * f3.y);
                    qq.x = half.x + c48 * (51.0 * fn.x + 3.0 * f1.x + f2.x);
                    qq.y = half.y + c48 * (51.0 * fn.y + 3.0 * f1.y + f2.y);
                    nw = cmk(pp.x - (161.0 / 170.0) * e.x, pp.y - (161.0 / 170.0) * e.y);
                    a.sC[o] = fn; a.sF[o] = nw; a.sG[o] = pp; a.sB[o] = qq;
                } else if (MODE == 2) {
                    const cplx w = a.W[o], m = a.sF[o], qq = a.sB[o], pp = a.sG[o];
                    const cplx fm = cmk((w.y - eta * m.y) * ih, -(w.x - eta * m.x) * ih);
                    const cplx cc = cmk(qq.x + c48 * 17.0 * fm.x, qq.y + c48 * 17.0 * fm.y);
                    const cplx ee = cmk(pp.x - cc.x, pp.y - cc.y);
                    nw = cmk(cc.x + (9.0 / 170.0) * ee.x, cc.y + (9.0 / 170.0) * ee.y);
                    a.sB[o] = nw; a.sF[o] = ee;
                } else {
                    const cplx w = a.W[o];
                    const cplx tt = (a.order == 1) ? a.sA[o] : a.sG[o];
                    const cplx gg = cmk((w.y - eta * tt.y) * ih, -(w.x - eta * tt.x) * ih);
                    const double cf = a.dt / (double)a.order;
                    const cplx tn = cmk(cf * gg.x, cf * gg.y);
                    a.sG[o] = tn;
                    if (a.order == 1) { if (a.write_f) a.sC[o] = gg; a.sF[o] = cadd(tt, tn); }
                    else a.sF[o] = cadd(a.sF[o], tn);
                    nw = tn;
                }
                if (cp == 0) nu0 = nw;
                if (cp >= 2) nv[cp - 2] = nw;
            }
            if (MODE != 3) {
                // pointwise densities: n (Eq. 3a), s = phi^+ sigma phi with phi = conj(v) (Eq. 3d), kappa (Eq. 3b)
                const cplx vu = nv[0], vd = nv[1];
                const double nu = vu.x * vu.x + vu.y * vu.y, nd = vd.x * vd.x + vd.y * vd.y;
                const double zr = vu.x * vd.x + vu.y * vd.y, zi = vu.y * vd.x - vu.x * vd.y;   // v_up conj(v_dn)
                dens[ACC_N * P + p] += nu + nd;
                dens[(ACC_S + 0) * P + p] += 2.0 * zr;
                dens[(ACC_S + 1) * P + p] += 2.0 * zi;
                dens[(ACC_S + 2) * P + p] += nu - nd;
                dens[(ACC_K + 0) * P + p] += vd.x * nu0.x + vd.y * nu0.y;      // conj(v_dn) u_up
                dens[(ACC_K + 1) * P + p] += vd.x * nu0.y - vd.y * nu0.x;
                phi[p] = cconj(vu); phi[P + p] = cconj(vd);
            }
        }
        if (MODE != 3) {
            __syncthreads();
            // y lines: LS = 1, PS = NZ; tasks = strips x {first-derivative, second-derivative}
            for (int task = warp; task < 2 * (NZ / 4); task += nwarps) {
                const int l0 = 4 * (task >> 1);
                if (task & 1) dens_axis_task<NY, 1>(phi, phi + P, dens, P, 1, l0, 1, NZ, s_cty);
                else          dens_axis_task<NY, 0>(phi, phi + P, dens, P, 1, l0, 1, NZ, s_cty);
            }
            __syncthreads();
            for (int task = warp; task < 2 * (NY / 4); task += nwarps) {
                const int l0 = 4 * (task >> 1);
                if (task & 1) dens_axis_task<NZ, 1>(phi, phi + P, dens, P, 2, l0, NZ, 1, s_ctz);
                else          dens_axis_task<NZ, 0>(phi, phi + P, dens, P, 2, l0, NZ, 1, s_ctz);
            }
            __syncthreads();
        }
    }
    if (MODE != 3) {
        double* part = a.part + (size_t)blockIdx.y * LISE_NACC * nxyz;
        for (int i = threadIdx.x; i < LISE_NACC * P; i += blockDim.x) {
            const int f = i / P, p = i - f * P;
            if (f == ACC_JC + 0) continue;                   // j_x comes from the x pass only
            part[(size_t)f * nxyz + gbase + p] += dens[i];
        }
    }
}

// x-axis density pass of the states in Z.   grid (ny, G), 256 threads.  shared: table | phi[2] | dens[5][P]
// local accumulator rows: 0 t, 1 j_x, 2 J_y (-= Xz), 3 J_z (+= Xy)  (axis 0 of dens_axis_task)
template <int NX>
__global__ void __launch_bounds__(256) k3_dens_x(DArgs a)
{
    extern __shared__ double2 smem[];
    const Lattice L = a.L;
    const int nz = L.nz, nxyz = L.nxyz, P = NX * nz, gs = L.ny * nz, gb = blockIdx.x * nz;
    double2* s_ctx = smem;
    cplx* phi = s_ctx + 2 * NX;
    double* dens = (double*)(phi + 2 * P);            // full LISE_NACC rows keep the indexing of dens_axis_task
    stage_table(s_ctx, a.ctab[0], NX);
    for (int i = threadIdx.x; i < LISE_NACC * P; i += blockDim.x) dens[i] = 0.0;
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    for (int st = blockIdx.y; st < a.ns; st += a.G) {
        const cplx* Zs = a.Z + (size_t)st * 4 * nxyz;
        __syncthreads();
        for (int p = threadIdx.x; p < P; p += blockDim.x) {
            const int ix = p / nz, iz = p - ix * nz, gi = gb + ix * gs + iz;
            phi[p] = cconj(Zs[(size_t)2 * nxyz + gi]); phi[P + p] = cconj(Zs[(size_t)3 * nxyz + gi]);
        }
        __syncthreads();
        for (int task = warp; task < 2 * (nz / 4); task += nwarps) {
            const int l0 = 4 * (task >> 1);
            if (task & 1) dens_axis_task<NX, 1>(phi, phi + P, dens, P, 0, l0, 1, nz, s_ctx);
            else          dens_axis_task<NX, 0>(phi, phi + P, dens, P, 0, l0, 1, nz, s_ctx);
        }
    }
    __syncthreads();
    double* part = a.part + (size_t)blockIdx.y * LISE_NACC * nxyz;
    const int rows[4] = {ACC_T, ACC_JC + 0, ACC_J + 1, ACC_J + 2};
    for (int i = threadIdx.x; i < 4 * P; i += blockDim.x) {
        const int k = i / P, p = i - k * P;
        const int ix = p / nz, iz = p - ix * nz, gi = gb + ix * gs + iz;
        part[(size_t)rows[k] * nxyz + gi] += dens[rows[k] * P + p];
    }
}
