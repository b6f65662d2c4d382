// state_kernels.cuh -- per-quasiparticle-state kernels: H-apply, ABM update, density accumulation.
//
// Decomposition used everywhere below: with
//   B_i = A_i 1 + (1/2)(sigma x W)_i   (2x2 Hermitian per point),
// the single-particle Hamiltonian of PAPER.md Eq. 12 in the lattice form of Eqs. 55-56 is
//   h = V_loc + sum_i T_i,   V_loc = U + (1/2) lap M + S.sigma,
//   T_i phi = -(1/2) [ M D2_i phi + D2_i (M phi) ] - i [ B_i D_i phi + D_i (B_i phi) ],
// and every T_i acts on independent lattice lines along axis i.  A CTA therefore works on one
// lattice PLANE staged in shared memory: yz-planes (contiguous in memory) carry the y and z lines,
// xz-planes carry the x lines.  D_i, D2_i are applied to a line as circulant sums with the
// closed-form DVR coefficients of PAPER.md Eq. 48 (generic DFMA line operator: any even lattice; the lattices the
// library is instantiated for run the tensor-core kernels of plane5_kernels.cuh instead).
#pragma once
#include "common.cuh"

// ------------------------------------------------------------------------------------------------
// line operator: circulant sums, register-blocked over R outputs per thread (lanes <-> lines)
//   MODE 0: dstA = D src, dstB = D2 src.      MODE 1: dstA += D srcA + D2 srcB.
// ct: shared-memory table, ct[N + d] = (c1[d mod N], c2[d mod N]) for d in (-N, N).
// ------------------------------------------------------------------------------------------------
template <int R, int MODE>
__device__ __forceinline__ void line_apply(const cplx* __restrict__ srcA, const cplx* __restrict__ srcB, int sstride,
                                           cplx* __restrict__ dstA, cplx* __restrict__ dstB, int dstride,
                                           int ncomp, int nlines, int N, int lstride, int pstride,
                                           const double2* __restrict__ ct)
{
    const int nblk = N / R;
    const int ntask = ncomp * nlines * nblk;
    for (int task = threadIdx.x; task < ntask; task += blockDim.x) {
        const int L = task % nlines;
        const int t2 = task / nlines;
        const int b = t2 % nblk;
        const int c = t2 / nblk;
        const int n0 = b * R;
        const cplx* xa = srcA + c * sstride + L * lstride;
        const cplx* xb = (MODE == 1) ? (srcB + c * sstride + L * lstride) : xa;
        const double2* cc = ct + N + n0;
        double ar[R], ai[R], br[R], bi[R];
#pragma unroll
        for (int r = 0; r < R; ++r) { ar[r] = 0.0; ai[r] = 0.0; br[r] = 0.0; bi[r] = 0.0; }
        for (int m = 0; m < N; ++m) {
            const cplx x = xa[m * pstride];
            cplx z = x;
            if (MODE == 1) z = xb[m * pstride];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double2 co = cc[r - m];
                if (MODE == 0) {
                    ar[r] = fma(co.x, x.x, ar[r]); ai[r] = fma(co.x, x.y, ai[r]);
                    br[r] = fma(co.y, x.x, br[r]); bi[r] = fma(co.y, x.y, bi[r]);
                } else {
                    ar[r] = fma(co.x, x.x, ar[r]); ai[r] = fma(co.x, x.y, ai[r]);
                    ar[r] = fma(co.y, z.x, ar[r]); ai[r] = fma(co.y, z.y, ai[r]);
                }
            }
        }
        cplx* da = dstA + c * dstride + L * lstride;
        if (MODE == 0) {
            cplx* db = dstB + c * dstride + L * lstride;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                da[(n0 + r) * pstride] = cmk(ar[r], ai[r]);
                db[(n0 + r) * pstride] = cmk(br[r], bi[r]);
            }
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                cplx o = da[(n0 + r) * pstride];
                da[(n0 + r) * pstride] = cmk(o.x + ar[r], o.y + ai[r]);
            }
        }
    }
}

// line-operator policies: the kernels below call LO::apply<MODE>(col_lines?, ...)
//   DenseLines<R>   : DFMA circulant sums, any even N (generic path)
//   (the fp64 tensor-core line operator lives in split_lineop.cuh / plane5_kernels.cuh and is not a policy of these kernels)
template <int R>
struct DenseLines {
    static constexpr int MAXT = 512;
    template <int MODE>
    static __device__ __forceinline__ void apply(bool col, const cplx* srcA, const cplx* srcB, int sstride,
                                                 cplx* dstA, cplx* dstB, int dstride, int ncomp,
                                                 int n1, int n2, int ld, const double2* ct)
    {
        if (col) line_apply<R, MODE>(srcA, srcB, sstride, dstA, dstB, dstride, ncomp, n2, n1, 1, ld, ct);
        else     line_apply<R, MODE>(srcA, srcB, sstride, dstA, dstB, dstride, ncomp, n1, n2, ld, 1, ct);
    }
};
// B_i = A_i + (1/2)(sigma x W)_i as (B00, B11, B01); B10 = conj(B01).   (from Eqs. 12, 56)
__device__ __forceinline__ void make_B(int axis, double A, double Wx, double Wy, double Wz,
                                       double& b00, double& b11, cplx& b01)
{
    if (axis == 0)      { b00 = A - 0.5 * Wy; b11 = A + 0.5 * Wy; b01 = cmk(0.0, -0.5 * Wz); }
    else if (axis == 1) { b00 = A + 0.5 * Wx; b11 = A - 0.5 * Wx; b01 = cmk(-0.5 * Wz, 0.0); }
    else                { b00 = A;            b11 = A;            b01 = cmk(0.5 * Wy, 0.5 * Wx); }
}
// (C in)_s with C = -i B
__device__ __forceinline__ void apply_C(double b00, double b11, cplx b01, cplx iu, cplx id, cplx& ou, cplx& od)
{
    cplx tu = cscale(b00, iu); cfma(tu, b01, id);
    cplx td = cscale(b11, id); cfma(td, cconj(b01), iu);
    ou = cmuli_neg(tu); od = cmuli_neg(td);
}

__device__ __forceinline__ double block_sum(double v, double* s_red)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (l == 0) s_red[w] = v;
    __syncthreads();
    double t = 0.0;
    for (int i = 0; i < nw; ++i) t += s_red[i];   // fixed order: deterministic
    return t;
}

__device__ __forceinline__ void stage_table(double2* s, const double2* __restrict__ g, int N)
{
    for (int i = threadIdx.x; i < 2 * N; i += blockDim.x) s[i] = g[i];
}

// ------------------------------------------------------------------------------------------------
// H-apply.  KIND 0 (yz-planes): W = [V_loc + T_y + T_z] X + pairing block.   grid (nx, G)
//           KIND 1 (xz-planes): W += T_x X, eta_part[st][iy] = dV Re <X|W> over the plane. grid (ny, G)
// Full state (Eq. 11, mu = 0): (H psi)_u = h u + Delta (v_dn, -v_up),
//                                       (H psi)_v = -conj(h conj v) + conj(Delta) (-u_dn, u_up).
// ------------------------------------------------------------------------------------------------
struct HArgs {
    alignas(64) CUtensorMap tmX;   // tensor map of X as [4 ns][nx][ny][2 nz doubles], 128-byte swizzled plane tiles (TMA kernels only)
    Lattice L;
    const cplx* X;
    cplx* W;
    const double* pot;        // [LISE_NPOT][nxyz]
    const double2* ctab[3];   // doubled circulant tables per axis (global; generic kernels)
    const double* stab[3];    // block-diagonalised tables per axis (split_lineop.cuh; plane5 kernels)
    double* eta_part;         // [ns][ny]
    int ns, G;
};

template <int KIND, class LO>
__global__ void __launch_bounds__(LO::MAXT) k_happly(HArgs a)
{
    extern __shared__ double2 smem[];
    const Lattice L = a.L;
    const Plane pl = make_plane(L, KIND, blockIdx.x);
    const int P = pl.n1 * pl.ld;
    const int npts = pl.npts();
    const int nxyz = L.nxyz;
    // shared layout: tables | phi[2] | ab[4] | out[2] | red
    double2* s_ctc = smem;                                   // column-line axis (y for KIND 0, x for KIND 1)
    double2* s_ctr = s_ctc + 2 * pl.n1;                      // row-line axis (z)
    cplx* phi = s_ctr + 2 * pl.n2;
    cplx* ab = phi + 2 * P;
    cplx* out = ab + 4 * P;
    double* s_red = (double*)(out + 2 * P);
    const int axc = (KIND == 0) ? 1 : 0;
    stage_table(s_ctc, a.ctab[axc], pl.n1);
    if (KIND == 0) stage_table(s_ctr, a.ctab[2], pl.n2);
    const double* pot = a.pot;

    for (int st = blockIdx.y; st < a.ns; st += a.G) {
        const cplx* Xs = a.X + (size_t)st * 4 * nxyz;
        cplx* Ws = a.W + (size_t)st * 4 * nxyz;
        double eta_loc = 0.0;
        for (int pair = 0; pair < 2; ++pair) {
            // ---- load the 2-spinor phi (pair 1: phi = conj(v)); initialise out ----
            for (int p = threadIdx.x; p < npts; p += blockDim.x) {
                const int r1 = p / pl.n2, c = p - r1 * pl.n2;
                const int si = r1 * pl.ld + c, gi = pl.gbase + r1 * pl.gs1 + c;
                cplx fu = Xs[(size_t)(2 * pair) * nxyz + gi], fd = Xs[(size_t)(2 * pair + 1) * nxyz + gi];
                if (pair) { fu = cconj(fu); fd = cconj(fd); }
                phi[si] = fu; phi[P + si] = fd;
                if (KIND == 0) {
                    const double ul = pot[(size_t)P_ULOC * nxyz + gi];
                    const double sx = pot[(size_t)(P_S + 0) * nxyz + gi], sy = pot[(size_t)(P_S + 1) * nxyz + gi],
                                 sz = pot[(size_t)(P_S + 2) * nxyz + gi];
                    // V_loc phi: (U + lap M / 2) phi + S.sigma phi
                    cplx ou = cscale(ul + sz, fu); cfma(ou, cmk(sx, -sy), fd);
                    cplx od = cscale(ul - sz, fd); cfma(od, cmk(sx, sy), fu);
                    out[si] = ou; out[P + si] = od;
                } else {
                    out[si] = cmk(0.0, 0.0); out[P + si] = cmk(0.0, 0.0);
                }
            }
            __syncthreads();
            // ---- the in-plane axes ----
            const int naxes = (KIND == 0) ? 2 : 1;
            for (int ia = 0; ia < naxes; ++ia) {
                // ia == 0: column lines (points along n1, stride ld); ia == 1: row lines (z)
                const int axis = (ia == 0) ? axc : 2;
                const double2* ct = (ia == 0) ? s_ctc : s_ctr;
                // a_s = D phi_s, b_s = D2 phi_s
                LO::template apply<0>(ia == 0, phi, phi, P, ab, ab + P, 2 * P, 2, pl.n1, pl.n2, pl.ld, ct);
                __syncthreads();
                for (int p = threadIdx.x; p < npts; p += blockDim.x) {
                    const int r1 = p / pl.n2, c = p - r1 * pl.n2;
                    const int si = r1 * pl.ld + c, gi = pl.gbase + r1 * pl.gs1 + c;
                    const double M = pot[(size_t)P_M * nxyz + gi];
                    const double A = pot[(size_t)(P_A + axis) * nxyz + gi];
                    const double Wx = pot[(size_t)(P_W + 0) * nxyz + gi], Wy = pot[(size_t)(P_W + 1) * nxyz + gi],
                                 Wz = pot[(size_t)(P_W + 2) * nxyz + gi];
                    double b00, b11; cplx b01;
                    make_B(axis, A, Wx, Wy, Wz, b00, b11, b01);
                    const cplx fu = phi[si], fd = phi[P + si];
                    const cplx au = ab[si], bu = ab[P + si], ad = ab[2 * P + si], bd = ab[3 * P + si];
                    cplx lu, ld_, gu, gd;
                    apply_C(b00, b11, b01, au, ad, lu, ld_);      // C D phi
                    caxpy(lu, -0.5 * M, bu); caxpy(ld_, -0.5 * M, bd);   // - M D2 phi / 2
                    cplx ou = out[si], od = out[P + si];
                    out[si] = cadd(ou, lu); out[P + si] = cadd(od, ld_);
                    apply_C(b00, b11, b01, fu, fd, gu, gd);       // g = C phi
                    ab[si] = gu; ab[P + si] = cscale(-0.5 * M, fu);            // q = -M phi / 2
                    ab[2 * P + si] = gd; ab[3 * P + si] = cscale(-0.5 * M, fd);
                }
                __syncthreads();
                // out_s += D g_s + D2 q_s
                LO::template apply<1>(ia == 0, ab, ab + P, 2 * P, out, out, P, 2, pl.n1, pl.n2, pl.ld, ct);
                __syncthreads();
            }
            // ---- write ----
            for (int p = threadIdx.x; p < npts; p += blockDim.x) {
                const int r1 = p / pl.n2, c = p - r1 * pl.n2;
                const int si = r1 * pl.ld + c, gi = pl.gbase + r1 * pl.gs1 + c;
                cplx ou = out[si], od = out[P + si];
                cplx* wu = Ws + (size_t)(2 * pair) * nxyz + gi;
                cplx* wd = Ws + (size_t)(2 * pair + 1) * nxyz + gi;
                if (KIND == 0) {
                    const cplx Dl = cmk(pot[(size_t)P_DELTA * nxyz + gi], pot[(size_t)(P_DELTA + 1) * nxyz + gi]);
                    if (pair == 0) {
                        const cplx vu = Xs[(size_t)2 * nxyz + gi], vd = Xs[(size_t)3 * nxyz + gi];
                        cfma(ou, Dl, vd);
                        cfma(od, cmk(-Dl.x, -Dl.y), vu);
                    } else {
                        const cplx uu = Xs[gi], ud = Xs[(size_t)nxyz + gi];
                        const cplx Dc = cconj(Dl);
                        ou = cmk(-ou.x, ou.y); od = cmk(-od.x, od.y);       // -conj(h conj v)
                        cfma(ou, cmk(-Dc.x, -Dc.y), ud);
                        cfma(od, Dc, uu);
                    }
                    *wu = ou; *wd = od;
                } else {
                    if (pair) { ou = cmk(-ou.x, ou.y); od = cmk(-od.x, od.y); }
                    const cplx tu = cadd(*wu, ou), td = cadd(*wd, od);
                    *wu = tu; *wd = td;
                    cplx xu = phi[si], xd = phi[P + si];
                    if (pair) { xu = cconj(xu); xd = cconj(xd); }
                    eta_loc += xu.x * tu.x + xu.y * tu.y + xd.x * td.x + xd.y * td.y;
                }
            }
            __syncthreads();
        }
        if (KIND == 1) {
            const double t = block_sum(eta_loc, s_red);
            if (threadIdx.x == 0) a.eta_part[(size_t)st * L.ny + blockIdx.x] = t * L.dV;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// density contributions of one axis at one point (Eq. 3 with phi = conj(v), tau via Eq. 51):
//   t += sum_s Re(phi_s^* D2_i phi_s),  j_i += sum_s Im(phi_s^* D_i phi_s),
//   J_k += eps_{kij} Im(phi^dagger sigma_j D_i phi)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dens_axis_rmw(double* part, int nxyz, int gi, int axis,
                                              cplx fu, cplx fd, cplx au, cplx ad, cplx bu, cplx bd)
{
    const double t = fu.x * bu.x + fu.y * bu.y + fd.x * bd.x + fd.y * bd.y;
    const double ji = (fu.x * au.y - fu.y * au.x) + (fd.x * ad.y - fd.y * ad.x);
    // z1 = conj(phi_up) a_dn, z2 = conj(phi_dn) a_up
    const double z1r = fu.x * ad.x + fu.y * ad.y, z1i = fu.x * ad.y - fu.y * ad.x;
    const double z2r = fd.x * au.x + fd.y * au.y, z2i = fd.x * au.y - fd.y * au.x;
    const double Xx = z1i + z2i;
    const double Xy = -z1r + z2r;
    const double Xz = (fu.x * au.y - fu.y * au.x) - (fd.x * ad.y - fd.y * ad.x);
    part[(size_t)ACC_T * nxyz + gi] += t;
    part[(size_t)(ACC_JC + axis) * nxyz + gi] += ji;
    if (axis == 0)      { part[(size_t)(ACC_J + 2) * nxyz + gi] += Xy; part[(size_t)(ACC_J + 1) * nxyz + gi] -= Xz; }
    else if (axis == 1) { part[(size_t)(ACC_J + 0) * nxyz + gi] += Xz; part[(size_t)(ACC_J + 2) * nxyz + gi] -= Xx; }
    else                { part[(size_t)(ACC_J + 1) * nxyz + gi] += Xx; part[(size_t)(ACC_J + 0) * nxyz + gi] -= Xy; }
}

// ------------------------------------------------------------------------------------------------
// ABM update fused with the y/z density pass of the NEW state.   grid (nx, G), yz-planes.
//   MODE 0: densities only of the states in Z.
//   MODE 1 (after evaluation 1, W = H y_n):  f_n = -i (W - eta y_n)/hbar c;
//            p = (y_n + y_{n-1})/2 + dt/48 (119 f_n - 99 f_{n-1} + 69 f_{n-2} - 17 f_{n-3})   (Eq. 78a)
//            m = p - 161/170 e_n                                                              (Eq. 78b)
//            Q = (y_n + y_{n-1})/2 + dt/48 (51 f_n + 3 f_{n-1} + f_{n-2})   [part of Eq. 78c]
//            writes f_n -> sC (was f_{n-3}), m -> sG, Q -> sB (was y_{n-1}); new state = m; e_n stays in sF
//   MODE 2 (after evaluation 2, W = H m):  m' = -i (W - eta m)/hbar c; c = Q + dt/48 17 m'    (Eq. 78c)
//            p = m + 161/170 e_n (Eq. 78b solved for p: p is not stored)
//            y_{n+1} = c + 9/170 (p - c) -> sB, e_{n+1} = p - c -> sF                          (Eq. 78d); new state = y_{n+1}
//   MODE 3 (series expansion, Eqs. 75-77): g = -i (W - eta T)/hbar c with T = sA (order 1) or sG;
//            order 1: eta fixed := eta_k, f_n = g -> sC, T' = dt g -> sG, acc = sA + T' -> sF
//            order m: T' = dt/m g -> sG, acc += T' -> sF;   no densities
// ------------------------------------------------------------------------------------------------
struct UArgs {
    Lattice L;
    const cplx* W;
    cplx *sA, *sB, *sC, *sD, *sE, *sF, *sG;   // chunk-offset slot pointers (roles, see above)
    const cplx* Z;                             // MODE 0 input
    const double* eta_part;                    // [ns][ny]
    double* eta_fix;                           // [ns]
    double* part;                              // [G][LISE_NACC][nxyz]
    const double2* ctab[3];
    double dt, hbarc;
    int ns, G, order, remove_phase, write_f;
    int neta;                                  // eta partial sums per state (v4 kernels; the generic ones use L.ny)
};

template <int MODE, class LO>
__global__ void __launch_bounds__(LO::MAXT) k_update_yz(UArgs a)
{
    extern __shared__ double2 smem[];
    const Lattice L = a.L;
    const Plane pl = make_plane(L, 0, blockIdx.x);
    const int P = pl.n1 * pl.ld;
    const int npts = pl.npts();
    const int nxyz = L.nxyz;
    double2* s_ctc = smem;
    double2* s_ctr = s_ctc + 2 * pl.n1;
    cplx* phi = s_ctr + 2 * pl.n2;
    cplx* ab = phi + 2 * P;
    double* s_eta = (double*)(ab + 4 * P);
    if (MODE != 3) { stage_table(s_ctc, a.ctab[1], pl.n1); stage_table(s_ctr, a.ctab[2], pl.n2); }
    double* part = a.part + (size_t)blockIdx.y * LISE_NACC * nxyz;
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
        for (int p = threadIdx.x; p < npts; p += blockDim.x) {
            const int r1 = p / pl.n2, c = p - r1 * pl.n2;
            const int si = r1 * pl.ld + c, gi = pl.gbase + r1 * pl.gs1 + c;
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
                    a.sC[o] = fn; a.sG[o] = nw; a.sB[o] = qq;
                } else if (MODE == 2) {
                    const cplx w = a.W[o], m = a.sG[o], qq = a.sB[o], en = a.sF[o];
                    const cplx pp = cmk(m.x + (161.0 / 170.0) * en.x, m.y + (161.0 / 170.0) * en.y);   // Eq. 78b solved for p
                    const cplx fm = cmk((w.y - eta * m.y) * ih, -(w.x - eta * m.x) * ih);
                    const cplx cc = cmk(qq.x + c48 * 17.0 * fm.x, qq.y + c48 * 17.0 * fm.y);
                    const cplx ee = cmk(pp.x - cc.x, pp.y - cc.y);
                    nw = cmk(cc.x + (9.0 / 170.0) * ee.x, cc.y + (9.0 / 170.0) * ee.y);
                    a.sB[o] = nw; a.sF[o] = ee;
                } else {
                    const cplx w = a.W[o];
                    const cplx t = (a.order == 1) ? a.sA[o] : a.sG[o];
                    const cplx g = cmk((w.y - eta * t.y) * ih, -(w.x - eta * t.x) * ih);
                    const double cf = a.dt / (double)a.order;
                    const cplx tn = cmk(cf * g.x, cf * g.y);
                    a.sG[o] = tn;
                    if (a.order == 1) { if (a.write_f) a.sC[o] = g; a.sF[o] = cadd(t, tn); }
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
                part[(size_t)ACC_N * nxyz + gi] += nu + nd;
                part[(size_t)(ACC_S + 0) * nxyz + gi] += 2.0 * zr;
                part[(size_t)(ACC_S + 1) * nxyz + gi] += 2.0 * zi;
                part[(size_t)(ACC_S + 2) * nxyz + gi] += nu - nd;
                part[(size_t)(ACC_K + 0) * nxyz + gi] += vd.x * nu0.x + vd.y * nu0.y;      // conj(v_dn) u_up
                part[(size_t)(ACC_K + 1) * nxyz + gi] += vd.x * nu0.y - vd.y * nu0.x;
                phi[si] = cconj(vu); phi[P + si] = cconj(vd);
            }
        }
        if (MODE != 3) {
            __syncthreads();
            for (int ia = 0; ia < 2; ++ia) {
                const int axis = (ia == 0) ? 1 : 2;
                const double2* ct = (ia == 0) ? s_ctc : s_ctr;
                LO::template apply<0>(ia == 0, phi, phi, P, ab, ab + P, 2 * P, 2, pl.n1, pl.n2, pl.ld, ct);
                __syncthreads();
                for (int p = threadIdx.x; p < npts; p += blockDim.x) {
                    const int r1 = p / pl.n2, c = p - r1 * pl.n2;
                    const int si = r1 * pl.ld + c, gi = pl.gbase + r1 * pl.gs1 + c;
                    dens_axis_rmw(part, nxyz, gi, axis, phi[si], phi[P + si], ab[si], ab[2 * P + si], ab[P + si], ab[3 * P + si]);
                }
                __syncthreads();
            }
        }
    }
}

// x-axis density pass of the states in Z.   grid (ny, G), xz-planes.
struct DArgs {
    Lattice L;
    const cplx* Z;
    double* part;
    const double2* ctab[3];
    const double* stab[3];
    int ns, G;
};
template <class LO>
__global__ void __launch_bounds__(LO::MAXT) k_dens_x(DArgs a)
{
    extern __shared__ double2 smem[];
    const Lattice L = a.L;
    const Plane pl = make_plane(L, 1, blockIdx.x);
    const int P = pl.n1 * pl.ld;
    const int npts = pl.npts();
    const int nxyz = L.nxyz;
    double2* s_ctc = smem;
    cplx* phi = s_ctc + 2 * pl.n1;
    cplx* ab = phi + 2 * P;
    stage_table(s_ctc, a.ctab[0], pl.n1);
    double* part = a.part + (size_t)blockIdx.y * LISE_NACC * nxyz;
    for (int st = blockIdx.y; st < a.ns; st += a.G) {
        const cplx* Zs = a.Z + (size_t)st * 4 * nxyz;
        __syncthreads();
        for (int p = threadIdx.x; p < npts; p += blockDim.x) {
            const int r1 = p / pl.n2, c = p - r1 * pl.n2;
            const int si = r1 * pl.ld + c, gi = pl.gbase + r1 * pl.gs1 + c;
            phi[si] = cconj(Zs[(size_t)2 * nxyz + gi]); phi[P + si] = cconj(Zs[(size_t)3 * nxyz + gi]);
        }
        __syncthreads();
        LO::template apply<0>(true, phi, phi, P, ab, ab + P, 2 * P, 2, pl.n1, pl.n2, pl.ld, s_ctc);
        __syncthreads();
        for (int p = threadIdx.x; p < npts; p += blockDim.x) {
            const int r1 = p / pl.n2, c = p - r1 * pl.n2;
            const int si = r1 * pl.ld + c, gi = pl.gbase + r1 * pl.gs1 + c;
            dens_axis_rmw(part, nxyz, gi, 0, phi[si], phi[P + si], ab[si], ab[2 * P + si], ab[P + si], ab[3 * P + si]);
        }
    }
}

// norms and sampled overlaps: out[(k*4 + t)] = dV <psi_k|psi_l>, l = k (t=0), k+1, k+2, k+nwf/2 (mod nwf)
static __global__ void k_overlaps(const cplx* __restrict__ Y, int nwf, int len, double dV, cplx* __restrict__ out)
{
    __shared__ double s_red[64];
    const int k = blockIdx.x, t = blockIdx.y;
    const int d = (t == 0) ? 0 : (t == 1) ? 1 : (t == 2) ? 2 : nwf / 2;
    const int l = (k + d) % nwf;
    const cplx* a = Y + (size_t)k * len;
    const cplx* b = Y + (size_t)l * len;
    double sr = 0.0, si = 0.0;
    for (int i = threadIdx.x; i < len; i += blockDim.x) {
        const cplx x = a[i], y = b[i];
        sr += x.x * y.x + x.y * y.y;
        si += x.x * y.y - x.y * y.x;
    }
    const double tr = block_sum(sr, s_red);
    const double ti = block_sum(si, s_red + 32);
    if (threadIdx.x == 0) out[k * 4 + t] = cmk(tr * dV, ti * dV);
}
