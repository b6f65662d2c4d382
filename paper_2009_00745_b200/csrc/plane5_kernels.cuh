// plane5_kernels.cuh -- the per-state kernels, "v5": block-diagonalised circulant line operator (split_lineop.cuh),
// DMMA-bound kernels and the HBM-bound ABM update separated so that each runs near its own roofline and the two
// classes can overlap on different streams.
//
//   k5_happly_yz : W  = [V_loc + T_y + T_z] X + pairing block     (yz-plane owner CTAs, X prefetched by cp.async)
//   k5_happly_xz : W += T_x X, eta partial sums                    (xz-plane owner CTAs)
//   k5_update    : f = -i (W - eta psi) / hbar c, Eq. 78  (pure streaming, no shared memory)
//   k5_dens_yz   : n, s, kappa pointwise + y/z-line parts of t, j, J of the new state (register accumulators)
//   k5_dens_x    : x-line parts of t, j, J of the new state
//
// Decomposition: h = V_loc + sum_i T_i,
//   T_i phi = -(1/2) [ M D2_i phi + D2_i (M phi) ] - i [ B_i D_i phi + D_i (B_i phi) ],  B_i = A_i + (sigma x W)_i / 2.
// A warp task = one 2-spinor on a strip of 4 lines (8 real DMMA columns: re | im of each line), all N outputs.
// Thread (g = lane / 4, t = lane % 4): feeds operand rows 4 kk + t (+ H m) of column g = (line l0 + g / 2, re | im),
// owns output rows 8 r + g (+ H m) of line l0 + t (accumulator columns 2 t, 2 t + 1 = re, im).
#pragma once
#include "common.cuh"
#include "state_kernels.cuh"
#include "plane_common.cuh"
#include "split_lineop.cuh"

__device__ __forceinline__ void bar_named(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// 8-byte part (re if !im, im if im) of a complex in shared memory
__device__ __forceinline__ double ld_part(const cplx* p, int idx, bool im) { return ((const double*)p)[2 * idx + (im ? 1 : 0)]; }
// x with its sign bit xor-ed by sgn (0 or 0x80000000): conjugation on the integer pipe, the fp64 pipe stays free
__device__ __forceinline__ double xor_sign(double x, unsigned sgn) { return __hiloint2double(__double2hiint(x) ^ (int)sgn, __double2loint(x)); }

// -i B a for the 2x2 Hermitian B = A + (sigma x W)_axis / 2 (compact potentials A, w1, w2 of AxisPot4), per axis
template <int AXIS>
__device__ __forceinline__ void apply_miB(double A, double w1, double w2, cplx au, cplx ad, cplx& ou, cplx& od)
{
    double tur, tui, tdr, tdi;
    if (AXIS == 0) {            // b00 = A - w1, b11 = A + w1, b01 = (0, beta), beta = -w2
        const double b00 = A - w1, b11 = A + w1;
        tur = fma(b00, au.x, w2 * ad.y);  tui = fma(b00, au.y, -w2 * ad.x);
        tdr = fma(b11, ad.x, -w2 * au.y); tdi = fma(b11, ad.y, w2 * au.x);
    } else if (AXIS == 1) {     // b00 = A + w1, b11 = A - w1, b01 = (alpha, 0), alpha = -w2
        const double b00 = A + w1, b11 = A - w1;
        tur = fma(b00, au.x, -w2 * ad.x); tui = fma(b00, au.y, -w2 * ad.y);
        tdr = fma(b11, ad.x, -w2 * au.x); tdi = fma(b11, ad.y, -w2 * au.y);
    } else {                    // b00 = b11 = A, b01 = (w1, w2)
        tur = fma(A, au.x, fma(w1, ad.x, -w2 * ad.y)); tui = fma(A, au.y, fma(w1, ad.y, w2 * ad.x));
        tdr = fma(A, ad.x, fma(w1, au.x, w2 * au.y));  tdi = fma(A, ad.y, fma(w1, au.y, -w2 * au.x));
    }
    ou = cmk(tui, -tur); od = cmk(tdi, -tdr);
}

template <int N> struct TaskGeom {
    typedef LOp<N> L;
    static constexpr int NA = L::R * L::NTH;      // output points per thread: index m * NTH + r <-> row H m + 8 r + g
};

// ------------------------------------------------------------------------------------------------
// T_axis phi of one 2-spinor on a strip of 4 lines -> registers (ru, rd)[m * NTH + r].
// CONJ: the planes hold raw v components; phi = conj(v) is formed on the fly.
// ------------------------------------------------------------------------------------------------
template <int N, int AXIS, bool CONJ>
__device__ __forceinline__ void taxis_core5(const cplx* __restrict__ phi_u, const cplx* __restrict__ phi_d, const AxisPot4 pot,
                                            int l0, int LS, int PS, const double* __restrict__ tab,
                                            cplx (&ru)[TaskGeom<N>::NA], cplx (&rd)[TaskGeom<N>::NA])
{
    typedef LOp<N> L;
    constexpr int R = L::R, NTH = L::NTH, NKH = L::NKH, H = L::H;
    constexpr bool SPLIT = (R * NTH >= 6);        // long lines: one operator at a time (register budget)
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const bool im = g & 1;
    const unsigned cs = (CONJ && im) ? 0x80000000u : 0u;   // sign flip of this lane's part under conjugation
    const int ibase = (l0 + (g >> 1)) * LS + t * PS;
    const int obase = (l0 + t) * LS + g * PS;
    // ---- phase 1: a = D phi, b = D2 phi; result = -i B a - M b / 2 ----
    {
        double au[R][NTH][2], ad[R][NTH][2], bu[R][NTH][2], bd[R][NTH][2];
        zero_acc<N>(au); zero_acc<N>(ad); zero_acc<N>(bu); zero_acc<N>(bd);
#pragma unroll
        for (int op = 0; op < (SPLIT ? 2 : 1); ++op) {
            Frags<N> F1, F2;
            if (!SPLIT || op == 0) F1.load(tab, 0, g, t);
            if (!SPLIT || op == 1) F2.load(tab, 1, g, t);
#pragma unroll
            for (int kk = 0; kk < NKH; ++kk) {
                double xu[R], xd[R], vu[R], vd[R];
#pragma unroll
                for (int m = 0; m < R; ++m) {
                    const int ii = ibase + (H * m + 4 * kk) * PS;
                    xu[m] = ld_part(phi_u, ii, im); xd[m] = ld_part(phi_d, ii, im);
                    if (CONJ) { xu[m] = xor_sign(xu[m], cs); xd[m] = xor_sign(xd[m], cs); }
                }
                RDFT<R>::fwd(xu, vu); RDFT<R>::fwd(xd, vd);
                if (!SPLIT || op == 0) { mma_blocks<N>(au, F1, vu, kk); mma_blocks<N>(ad, F1, vd, kk); }
                if (!SPLIT || op == 1) { mma_blocks<N>(bu, F2, vu, kk); mma_blocks<N>(bd, F2, vd, kk); }
            }
        }
        post_transform<N>(au); post_transform<N>(ad); post_transform<N>(bu); post_transform<N>(bd);
#pragma unroll
        for (int m = 0; m < R; ++m)
#pragma unroll
            for (int r = 0; r < NTH; ++r) {
                const int idx = m * NTH + r;
                if (8 * r + g >= H) { ru[idx] = cmk(0.0, 0.0); rd[idx] = cmk(0.0, 0.0); continue; }   // padding rows
                const int oi = obase + (H * m + 8 * r) * PS;
                const double mh = pot.M[oi];                                       // -M / 2
                cplx lu, ld_;
                apply_miB<AXIS>(pot.A[oi], pot.w1[oi], pot.w2[oi], cmk(au[m][r][0], au[m][r][1]), cmk(ad[m][r][0], ad[m][r][1]), lu, ld_);   // -i B D phi
                ru[idx] = cmk(fma(mh, bu[m][r][0], lu.x), fma(mh, bu[m][r][1], lu.y));
                rd[idx] = cmk(fma(mh, bd[m][r][0], ld_.x), fma(mh, bd[m][r][1], ld_.y));
            }
    }
    // ---- phase 2: c = D g + D2 q,  g = -i B phi,  q = -M phi / 2 ----
    {
        double cu[R][NTH][2], cd[R][NTH][2];
        zero_acc<N>(cu); zero_acc<N>(cd);
#pragma unroll
        for (int op = 0; op < (SPLIT ? 2 : 1); ++op) {
            Frags<N> F1, F2;
            if (!SPLIT || op == 0) F1.load(tab, 0, g, t);
            if (!SPLIT || op == 1) F2.load(tab, 1, g, t);
#pragma unroll
            for (int kk = 0; kk < NKH; ++kk) {
                double gu[R], gd[R], qu[R], qd[R];
#pragma unroll
                for (int m = 0; m < R; ++m) {
                    const int ii = ibase + (H * m + 4 * kk) * PS;
                    cplx fu = phi_u[ii], fd = phi_d[ii];
                    if (CONJ) { fu.y = xor_sign(fu.y, 0x80000000u); fd.y = xor_sign(fd.y, 0x80000000u); }
                    if (!SPLIT || op == 0) g_part4<AXIS>(im, pot.A[ii], pot.w1[ii], pot.w2[ii], fu, fd, gu[m], gd[m]);
                    if (!SPLIT || op == 1) {
                        const double mh = pot.M[ii];                                   // -M / 2
                        qu[m] = mh * (im ? fu.y : fu.x); qd[m] = mh * (im ? fd.y : fd.x);
                    }
                }
                if (!SPLIT || op == 0) {
                    double vu[R], vd[R];
                    RDFT<R>::fwd(gu, vu); RDFT<R>::fwd(gd, vd);
                    mma_blocks<N>(cu, F1, vu, kk); mma_blocks<N>(cd, F1, vd, kk);
                }
                if (!SPLIT || op == 1) {
                    double vu[R], vd[R];
                    RDFT<R>::fwd(qu, vu); RDFT<R>::fwd(qd, vd);
                    mma_blocks<N>(cu, F2, vu, kk); mma_blocks<N>(cd, F2, vd, kk);
                }
            }
        }
        post_transform<N>(cu); post_transform<N>(cd);
#pragma unroll
        for (int m = 0; m < R; ++m)
#pragma unroll
            for (int r = 0; r < NTH; ++r) {
                const int idx = m * NTH + r;
                ru[idx].x += cu[m][r][0]; ru[idx].y += cu[m][r][1];
                rd[idx].x += cd[m][r][0]; rd[idx].y += cd[m][r][1];
            }
    }
}

// ------------------------------------------------------------------------------------------------
// H-apply, yz-planes:  W = [V_loc + T_y + T_z] X + pairing block (Eq. 11, mu = 0).
// grid (nx, G), NWARP warps.  A unit = NCOMP components (4: a state, 2: one 2-spinor) on the plane.
// Per unit: [cp.async wait + barrier] -> y tasks (result -> out planes) -> per-pair named barrier -> z tasks, whose
// epilogue adds the y result, V_loc phi, the pairing block, maps the v pair back (-conj) and stores W to global.
// shared: tables | phi[NBUF][NCOMP][PP] | out[NCOMP][PP] | pots M, Ay, Az, hWx, hWy, hWz [PP] | pV[6][PP] (VSTAGE)
// ------------------------------------------------------------------------------------------------
template <int NY, int NZ, int NCOMP, int NBUF, int NWARP, bool VSTAGE, int MAXR>
__global__ void __maxnreg__(MAXR) k5_happly_yz(HArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int LD = ldpad(NZ), PP = NY * LD, NPTS = NY * NZ;
    constexpr int NPAIR = NCOMP / 2, UPS = 4 / NCOMP;
    constexpr int WPP = NWARP / NPAIR;                      // warps per pair
    static_assert(NWARP % NPAIR == 0, "warps must split evenly over the pairs");
    const int nxyz = a.L.nxyz;
    const int gbase = blockIdx.x * NPTS;
    double* s_ty = (double*)smem;
    double* s_tz = s_ty + LOp<NY>::TABSZ;
    cplx* phi = (cplx*)(s_tz + LOp<NZ>::TABSZ + ((LOp<NY>::TABSZ + LOp<NZ>::TABSZ) & 1));
    cplx* out = phi + NBUF * NCOMP * PP;
    double* pM = (double*)(out + NCOMP * PP);
    double *pAy = pM + PP, *pAz = pAy + PP, *pWx = pAz + PP, *pWy = pWx + PP, *pWz = pWy + PP;
    double* pV = pWz + PP;
    const double* pot = a.pot;
    for (int i = threadIdx.x; i < LOp<NY>::TABSZ; i += blockDim.x) s_ty[i] = a.stab[1][i];
    for (int i = threadIdx.x; i < LOp<NZ>::TABSZ; i += blockDim.x) s_tz[i] = a.stab[2][i];
    auto stage_pots = [&]() {
    for (int p = threadIdx.x; p < NPTS; p += blockDim.x) {
        const int y = p / NZ, z = p - y * NZ, si = y * LD + z, gi = gbase + p;
        pM[si] = -0.5 * pot[(size_t)P_M * nxyz + gi];
        pAy[si] = pot[(size_t)(P_A + 1) * nxyz + gi]; pAz[si] = pot[(size_t)(P_A + 2) * nxyz + gi];
        pWx[si] = 0.5 * pot[(size_t)(P_W + 0) * nxyz + gi]; pWy[si] = 0.5 * pot[(size_t)(P_W + 1) * nxyz + gi];
        pWz[si] = 0.5 * pot[(size_t)(P_W + 2) * nxyz + gi];
        if (VSTAGE) {
            double v[6]; load_vloc(pot, nxyz, gi, v);
#pragma unroll
            for (int k = 0; k < 6; ++k) pV[k * PP + si] = v[k];
        }
    }
    };
    const AxisPot4 poty = {pM, pAy, pWx, pWz}, potz = {pM, pAz, pWy, pWx};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int pr = warp / WPP, lw = warp - pr * WPP;        // this warp's pair (within the unit) and index in it
    const int nunits = a.ns * UPS;
    // ASYNC (two X buffers): no CTA-wide barrier inside the unit loop.  mbarriers F[buf] ("unit landed": every thread's
    // cp.async copies arrive on it), E[buf] ("everyone is done with the unit in buf": out planes and X[buf] are free),
    // Y[pair] ("the pair's y results are in the out planes").  Waits sit behind a DMMA pass, so warps drift by up to a
    // task instead of stopping together.
    constexpr bool ASYNC = (NBUF == 2);
    __shared__ unsigned long long s_bar[6];
    unsigned long long *barF = s_bar, *barE = s_bar + 2, *barY = s_bar + 4;
    if (ASYNC) {
        if (threadIdx.x == 0) {
            mbar_init(barF, NWARP * 32); mbar_init(barF + 1, NWARP * 32);
            mbar_init(barE, NWARP * 32); mbar_init(barE + 1, NWARP * 32);
            mbar_init(barY, WPP * 32); mbar_init(barY + 1, WPP * 32);
        }
        __syncthreads();
    }

    auto issue = [&](int u, int buf) {
        const int st = u / UPS, pg = u - st * UPS;
        const cplx* Xs = a.X + ((size_t)st * 4 + pg * NCOMP) * nxyz + gbase;
        cplx* dst = phi + buf * NCOMP * PP;
        for (int i = threadIdx.x; i < NCOMP * NPTS; i += blockDim.x) {
            const int c = i / NPTS, p = i - c * NPTS, y = p / NZ, z = p - y * NZ;
            cp_async16(dst + c * PP + y * LD + z, Xs + (size_t)c * nxyz + p);
        }
        if (ASYNC) mbar_arrive_cp_async(barF + buf); else cp_async_commit();
    };

    int u = blockIdx.y;
    if (u < nunits) issue(u, 0);
    stage_pots();                                           // behind the first prefetch
    if (ASYNC) __syncthreads();                             // potentials and tables staged
    for (int it = 0; u < nunits; u += a.G, ++it) {
        const int buf = (NBUF == 2) ? (it & 1) : 0;
        if (ASYNC) mbar_wait(barF + buf, (it >> 1) & 1);    // unit u has landed
        else { cp_async_wait<0>(); __syncthreads(); }       // ... and everyone is done with unit u - G
        const int st = u / UPS, pg = u - st * UPS;
        const int pair = pg * NPAIR + pr;                   // 0: u pair, 1: v pair
        const cplx* phib = phi + buf * NCOMP * PP;
        const cplx *fu = phib + 2 * pr * PP, *fd = fu + PP;
        cplx *ou = out + 2 * pr * PP, *od = ou + PP;
        bool mid_done = false;
        auto mid_unit = [&]() {                             // once per unit and thread, behind the first y pass
            if (!ASYNC || mid_done) return;
            mid_done = true;
            if (it >= 1) mbar_wait(barE + (buf ^ 1), ((it - 1) >> 1) & 1);   // unit u - G: out planes and X[buf ^ 1] are free
            if (u + a.G < nunits) issue(u + a.G, buf ^ 1);
        };
        // ---- y lines (one per z): LS = 1, PS = LD; result -> out planes ----
        for (int task = lw; task < NZ / 4; task += WPP) {
            const int l0 = 4 * task;
            cplx ru[TaskGeom<NY>::NA], rd[TaskGeom<NY>::NA];
            if (pair) taxis_core5<NY, 1, true>(fu, fd, poty, l0, 1, LD, s_ty, ru, rd);
            else      taxis_core5<NY, 1, false>(fu, fd, poty, l0, 1, LD, s_ty, ru, rd);
            mid_unit();
            typedef LOp<NY> L;
#pragma unroll
            for (int m = 0; m < L::R; ++m)
#pragma unroll
                for (int r = 0; r < L::NTH; ++r) {
                    if (8 * r + g >= L::H) continue;
                    const int oi = (l0 + t) + (L::H * m + 8 * r + g) * LD;
                    ou[oi] = ru[m * L::NTH + r]; od[oi] = rd[m * L::NTH + r];
                }
        }
        mid_unit();
        if (ASYNC) mbar_arrive(barY + pr);                  // this thread's y results are in the out planes
        else bar_named(1 + pr, WPP * 32);                   // the pair's y results are complete
        bool y_waited = false;
        // ---- z lines (one per y): LS = LD, PS = 1; epilogue finishes W ----
        cplx* Ws = a.W + (size_t)st * 4 * nxyz;
        const cplx* Xst = a.X + (size_t)st * 4 * nxyz;
        for (int task = lw; task < NY / 4; task += WPP) {
            const int l0 = 4 * task;
            cplx ru[TaskGeom<NZ>::NA], rd[TaskGeom<NZ>::NA];
            if (pair) taxis_core5<NZ, 2, true>(fu, fd, potz, l0, LD, 1, s_tz, ru, rd);
            else      taxis_core5<NZ, 2, false>(fu, fd, potz, l0, LD, 1, s_tz, ru, rd);
            if (ASYNC && !y_waited) { mbar_wait(barY + pr, it & 1); y_waited = true; }   // behind the z pass: nobody waits
            typedef LOp<NZ> L;
#pragma unroll
            for (int m = 0; m < L::R; ++m)
#pragma unroll
                for (int r = 0; r < L::NTH; ++r) {
                    if (8 * r + g >= L::H) continue;
                    const int y = l0 + t, z = L::H * m + 8 * r + g;
                    const int si = y * LD + z, gi = gbase + y * NZ + z;
                    double v[6];
                    if (VSTAGE) {
#pragma unroll
                        for (int k = 0; k < 6; ++k) v[k] = pV[k * PP + si];
                    } else load_vloc(pot, nxyz, gi, v);
                    const double ul = v[0], sx = v[1], sy = v[2], sz = v[3];
                    const cplx Dl = cmk(v[4], v[5]);
                    cplx pu = fu[si], pd = fd[si];
                    if (pair) { pu = cconj(pu); pd = cconj(pd); }
                    cplx wu = cadd(ru[m * L::NTH + r], ou[si]), wd = cadd(rd[m * L::NTH + r], od[si]);
                    caxpy(wu, ul + sz, pu); cfma(wu, cmk(sx, -sy), pd);
                    caxpy(wd, ul - sz, pd); cfma(wd, cmk(sx, sy), pu);
                    if (pair == 0) {
                        cplx vu, vd;
                        if (NCOMP == 4) { vu = phib[2 * PP + si]; vd = phib[3 * PP + si]; }
                        else { vu = Xst[(size_t)2 * nxyz + gi]; vd = Xst[(size_t)3 * nxyz + gi]; }
                        cfma(wu, Dl, vd);
                        cfma(wd, cmk(-Dl.x, -Dl.y), vu);
                    } else {
                        cplx uu, ud;
                        if (NCOMP == 4) { uu = phib[si]; ud = phib[PP + si]; }
                        else { uu = Xst[gi]; ud = Xst[(size_t)nxyz + gi]; }
                        const cplx Dc = cconj(Dl);
                        wu = cmk(-wu.x, wu.y); wd = cmk(-wd.x, wd.y);           // -conj(h conj v)
                        cfma(wu, cmk(-Dc.x, -Dc.y), ud);
                        cfma(wd, Dc, uu);
                    }
                    Ws[(size_t)(2 * pair) * nxyz + gi] = wu; Ws[(size_t)(2 * pair + 1) * nxyz + gi] = wd;
                }
        }
        if (ASYNC) mbar_arrive(barE + buf);                 // this thread is done with unit u
        if (NBUF == 1) { __syncthreads(); if (u + a.G < nunits) issue(u + a.G, 0); }
    }
}

// ------------------------------------------------------------------------------------------------
// H-apply, xz-planes:  W += T_x X,  eta_part[(st * UPS + pg) * ny + iy] = dV Re <X|W> over the plane.
// grid (ny, G), NWARP warps.  One barrier per unit; the W values of a thread's output points are read from global
// before the DMMA passes and consumed in the epilogue.
// shared: table | phi[NBUF][NCOMP][PP] | w[NBUF][NCOMP][PP] (WST) | pots M, Ax, hWy, hWz [PP] | red[2][NWARP]
// ------------------------------------------------------------------------------------------------
template <int NX, int NZ, int NCOMP, int NBUF, int NWARP, int MAXR, bool WST>
__global__ void __maxnreg__(MAXR) k5_happly_xz(HArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int LD = ldpad(NZ), PP = NX * LD, NPTS = NX * NZ;
    constexpr int NPAIR = NCOMP / 2, UPS = 4 / NCOMP;
    typedef LOp<NX> L;
    constexpr int NA = TaskGeom<NX>::NA;
    const int nxyz = a.L.nxyz, gs = a.L.ny * NZ, gb = blockIdx.x * NZ;
    double* s_tx = (double*)smem;
    cplx* phi = (cplx*)(s_tx + L::TABSZ + (L::TABSZ & 1));
    cplx* wpl = phi + NBUF * NCOMP * PP;                    // WST: the unit's W plane, prefetched with its X plane
    double* pM = (double*)(wpl + (WST ? NBUF * NCOMP * PP : 0));
    double *pAx = pM + PP, *pWy = pAx + PP, *pWz = pWy + PP;
    double* s_red = pWz + PP;                               // [2][NWARP]
    const double* pot = a.pot;
    for (int i = threadIdx.x; i < L::TABSZ; i += blockDim.x) s_tx[i] = a.stab[0][i];
    auto stage_pots = [&]() {
    for (int p = threadIdx.x; p < NPTS; p += blockDim.x) {
        const int x = p / NZ, z = p - x * NZ, si = x * LD + z, gi = gb + x * gs + z;
        pM[si] = -0.5 * pot[(size_t)P_M * nxyz + gi];
        pAx[si] = pot[(size_t)(P_A + 0) * nxyz + gi];
        pWy[si] = 0.5 * pot[(size_t)(P_W + 1) * nxyz + gi]; pWz[si] = 0.5 * pot[(size_t)(P_W + 2) * nxyz + gi];
    }
    };
    const AxisPot4 potx = {pM, pAx, pWy, pWz};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int nunits = a.ns * UPS;

    // ASYNC: mbarriers F[buf] ("unit landed") and E[buf] ("everyone is done with the unit in buf") instead of a CTA-wide
    // barrier per unit; see k5_happly_yz.  Off: with one task per warp and unit the prefetch would be issued behind
    // that task and land too late (measured: 17.6 ms against 14.8 ms per step on config 1).
    constexpr bool ASYNC = false;
    __shared__ unsigned long long s_bar[4];
    unsigned long long *barF = s_bar, *barE = s_bar + 2;
    if (ASYNC) {
        if (threadIdx.x == 0) {
            mbar_init(barF, NWARP * 32); mbar_init(barF + 1, NWARP * 32);
            mbar_init(barE, NWARP * 32); mbar_init(barE + 1, NWARP * 32);
        }
        __syncthreads();
    }
    auto issue = [&](int u, int buf) {
        const int st = u / UPS, pg = u - st * UPS;
        const size_t go = ((size_t)st * 4 + pg * NCOMP) * nxyz + gb;
        cplx* dphi = phi + buf * NCOMP * PP;
        cplx* dw = wpl + buf * NCOMP * PP;
        for (int i = threadIdx.x; i < NCOMP * NPTS; i += blockDim.x) {
            const int c = i / NPTS, p = i - c * NPTS, x = p / NZ, z = p - x * NZ;
            const size_t gi = go + (size_t)c * nxyz + (size_t)x * gs + z;
            cp_async16(dphi + c * PP + x * LD + z, a.X + gi);
            if (WST) cp_async16(dw + c * PP + x * LD + z, a.W + gi);
        }
        if (ASYNC) mbar_arrive_cp_async(barF + buf); else cp_async_commit();
    };
    auto flush_eta = [&](int uprev, int it_prev) {          // thread 0: fixed-order sum of the warps' partials
        const int st = uprev / UPS, pg = uprev - st * UPS;
        double s = 0.0;
        for (int w = 0; w < NWARP; ++w) s += s_red[(it_prev & 1) * NWARP + w];
        a.eta_part[((size_t)st * UPS + pg) * a.L.ny + blockIdx.x] = s * a.L.dV;
    };

    int u = blockIdx.y, uprev = -1;
    if (u < nunits) issue(u, 0);
    stage_pots();                                           // behind the first prefetch
    if (ASYNC) __syncthreads();
    int it = 0;
    for (; u < nunits; u += a.G, ++it) {
        const int buf = (NBUF == 2) ? (it & 1) : 0;
        if (ASYNC) mbar_wait(barF + buf, (it >> 1) & 1);
        else {
            cp_async_wait<0>();
            __syncthreads();
            if (NBUF == 2 && u + a.G < nunits) issue(u + a.G, buf ^ 1);
            if (threadIdx.x == 0 && uprev >= 0) flush_eta(uprev, it - 1);
        }
        bool mid_done = false;
        auto mid_unit = [&]() {                             // once per unit and thread, behind the first x pass
            if (!ASYNC || mid_done) return;
            mid_done = true;
            if (it >= 1) {
                mbar_wait(barE + (buf ^ 1), ((it - 1) >> 1) & 1);       // everyone is done with unit u - G
                if (threadIdx.x == 0) flush_eta(uprev, it - 1);
            }
            if (u + a.G < nunits) issue(u + a.G, buf ^ 1);
        };
        const int st = u / UPS, pg = u - st * UPS;
        const cplx* phib = phi + buf * NCOMP * PP;
        double eta_loc = 0.0;
        // ---- x lines (one per z): LS = 1, PS = LD ----
        for (int task = warp; task < NPAIR * (NZ / 4); task += NWARP) {
            const int pr = task / (NZ / 4), l0 = 4 * (task - pr * (NZ / 4));
            const int pair = pg * NPAIR + pr;
            const cplx *fu = phib + 2 * pr * PP, *fd = fu + PP;
            cplx* Wu = a.W + ((size_t)st * 4 + 2 * pair) * nxyz + gb;
            cplx* Wd = Wu + nxyz;
            const cplx *swu = wpl + (buf * NCOMP + 2 * pr) * PP, *swd = swu + PP;
            cplx wu[WST ? 1 : NA], wd[WST ? 1 : NA];
            if (!WST) {
#pragma unroll
                for (int m = 0; m < L::R; ++m)
#pragma unroll
                    for (int r = 0; r < L::NTH; ++r) {
                        const int idx = m * L::NTH + r;
                        if (8 * r + g >= L::H) { wu[idx] = cmk(0.0, 0.0); wd[idx] = cmk(0.0, 0.0); continue; }
                        const size_t go = (size_t)(L::H * m + 8 * r + g) * gs + (l0 + t);
                        wu[idx] = Wu[go]; wd[idx] = Wd[go];
                    }
            }
            cplx ru[NA], rd[NA];
            if (pair) taxis_core5<NX, 0, true>(fu, fd, potx, l0, 1, LD, s_tx, ru, rd);
            else      taxis_core5<NX, 0, false>(fu, fd, potx, l0, 1, LD, s_tx, ru, rd);
            mid_unit();
#pragma unroll
            for (int m = 0; m < L::R; ++m)
#pragma unroll
                for (int r = 0; r < L::NTH; ++r) {
                    const int idx = m * L::NTH + r;
                    if (8 * r + g >= L::H) continue;
                    const int x = L::H * m + 8 * r + g, z = l0 + t;
                    cplx fu_ = WST ? swu[x * LD + z] : wu[idx], fd_ = WST ? swd[x * LD + z] : wd[idx];
                    if (pair) { fu_ = cmk(fu_.x - ru[idx].x, fu_.y + ru[idx].y); fd_ = cmk(fd_.x - rd[idx].x, fd_.y + rd[idx].y); }
                    else      { fu_ = cadd(fu_, ru[idx]); fd_ = cadd(fd_, rd[idx]); }
                    const size_t go = (size_t)x * gs + z;
                    Wu[go] = fu_; Wd[go] = fd_;
                    const cplx xu = fu[x * LD + z], xd = fd[x * LD + z];          // raw components
                    eta_loc += xu.x * fu_.x + xu.y * fu_.y + xd.x * fd_.x + xd.y * fd_.y;
                }
        }
        for (int o = 16; o > 0; o >>= 1) eta_loc += __shfl_xor_sync(0xffffffffu, eta_loc, o);
        mid_unit();
        if (lane == 0) s_red[(it & 1) * NWARP + warp] = eta_loc;
        if (ASYNC) mbar_arrive(barE + buf);
        uprev = u;
        if (NBUF == 1) { __syncthreads(); if (u + a.G < nunits) issue(u + a.G, 0); }
    }
    __syncthreads();
    if (threadIdx.x == 0 && uprev >= 0) flush_eta(uprev, it - 1);
}

// ------------------------------------------------------------------------------------------------
// ABM update, pure streaming (Eq. 78, Eqs. 80-81).  grid (blocks over the 4 nxyz elements of a state, ns).
//   MODE 1 (after evaluation 1): f_n = -i (W - eta y_n) / hbar c;  p, Q, m = p - (161/170) e;  C <- f_n, G <- m, B <- Q
//   MODE 2 (after evaluation 2): f_m; c = Q + (dt/48) 17 f_m; p = m + (161/170) e; e' = p - c; y_{n+1} = c + (9/170) e';
//           B <- y_{n+1}, F <- e'.   The predictor p is not stored: Eq. 78b is solved for it (one rounding), which saves
//           one of the 17 array passes of a step.
//   MODE 3 (starter, Taylor term `order`): as k_update_yz<3> in state_kernels.cuh
// History slots are read and written with streaming cache hints so that W, X and the new state stay in L2.
// ------------------------------------------------------------------------------------------------
// 128 threads (one warp per SM sub-partition) and <= LISE_UPD_REGS registers: one CTA fits beside a plane-owner CTA
// capped at coresident_regs() registers on the same SM, so the update of chunk i streams from HBM while the x-line
// H-apply and the density kernels of the neighbouring chunks run.
#define LISE_UPD_THREADS 128
template <int MODE> struct UpdEpt { static constexpr int V = (MODE == 1) ? 2 : (MODE == 2) ? 4 : 2; };   // elements per thread
template <int MODE>
__global__ void __maxnreg__(LISE_UPD_REGS) k5_update(UArgs a)
{
    __shared__ double s_eta;
    const int st = blockIdx.y;
    const size_t slen = (size_t)4 * a.L.nxyz;
    if (threadIdx.x == 0) {
        double eta = 0.0;
        if (MODE == 3 && a.order > 1) eta = a.eta_fix[st];
        else {
            for (int j = 0; j < a.neta; ++j) eta += a.eta_part[(size_t)st * a.neta + j];   // fixed order
            if (!a.remove_phase) eta = 0.0;
            if (MODE == 3 && blockIdx.x == 0) a.eta_fix[st] = eta;
        }
        s_eta = eta;
    }
    __syncthreads();
    const double eta = s_eta;
    const double ih = 1.0 / a.hbarc, c48 = a.dt / 48.0;
    const size_t so = (size_t)st * slen;
    constexpr int LISE_UPD_EPT = UpdEpt<MODE>::V;
    const size_t e0 = (size_t)blockIdx.x * (LISE_UPD_THREADS * LISE_UPD_EPT) + threadIdx.x;
    if (MODE == 1) {
        cplx w[LISE_UPD_EPT], y[LISE_UPD_EPT], ym[LISE_UPD_EPT], f1[LISE_UPD_EPT], f2[LISE_UPD_EPT], f3[LISE_UPD_EPT], e[LISE_UPD_EPT];
#pragma unroll
        for (int k = 0; k < LISE_UPD_EPT; ++k) {
            const size_t el = e0 + (size_t)k * LISE_UPD_THREADS;
            if (el >= slen) continue;
            const size_t o = so + el;
            w[k] = __ldcs(a.W + o); y[k] = __ldcs(a.sA + o); ym[k] = __ldcs(a.sB + o);
            f1[k] = __ldcs(a.sD + o); f2[k] = __ldcs(a.sE + o); f3[k] = __ldcs(a.sC + o); e[k] = __ldcs(a.sF + o);
        }
#pragma unroll
        for (int k = 0; k < LISE_UPD_EPT; ++k) {
            const size_t el = e0 + (size_t)k * LISE_UPD_THREADS;
            if (el >= slen) continue;
            const size_t o = so + el;
            const cplx fn = cmk((w[k].y - eta * y[k].y) * ih, -(w[k].x - eta * y[k].x) * ih);
            const cplx half = cmk(0.5 * (y[k].x + ym[k].x), 0.5 * (y[k].y + ym[k].y));
            cplx pp, qq;
            pp.x = half.x + c48 * (119.0 * fn.x - 99.0 * f1[k].x + 69.0 * f2[k].x - 17.0 * f3[k].x);
            pp.y = half.y + c48 * (119.0 * fn.y - 99.0 * f1[k].y + 69.0 * f2[k].y - 17.0 * f3[k].y);
            qq.x = half.x + c48 * (51.0 * fn.x + 3.0 * f1[k].x + f2[k].x);
            qq.y = half.y + c48 * (51.0 * fn.y + 3.0 * f1[k].y + f2[k].y);
            const cplx m = cmk(pp.x - (161.0 / 170.0) * e[k].x, pp.y - (161.0 / 170.0) * e[k].y);
            __stcs(a.sC + o, fn); __stcs(a.sB + o, qq);
            a.sG[o] = m;                                    // the new state: read again by the density kernels
        }
    } else if (MODE == 2) {
        cplx w[LISE_UPD_EPT], m[LISE_UPD_EPT], qq[LISE_UPD_EPT], en[LISE_UPD_EPT];
#pragma unroll
        for (int k = 0; k < LISE_UPD_EPT; ++k) {
            const size_t el = e0 + (size_t)k * LISE_UPD_THREADS;
            if (el >= slen) continue;
            const size_t o = so + el;
            w[k] = __ldcs(a.W + o); m[k] = __ldcs(a.sG + o); qq[k] = __ldcs(a.sB + o); en[k] = __ldcs(a.sF + o);
        }
#pragma unroll
        for (int k = 0; k < LISE_UPD_EPT; ++k) {
            const size_t el = e0 + (size_t)k * LISE_UPD_THREADS;
            if (el >= slen) continue;
            const size_t o = so + el;
            const cplx fm = cmk((w[k].y - eta * m[k].y) * ih, -(w[k].x - eta * m[k].x) * ih);
            const cplx cc = cmk(qq[k].x + c48 * 17.0 * fm.x, qq[k].y + c48 * 17.0 * fm.y);
            const cplx pp = cmk(m[k].x + (161.0 / 170.0) * en[k].x, m[k].y + (161.0 / 170.0) * en[k].y);   // Eq. 78b solved for p
            const cplx ee = cmk(pp.x - cc.x, pp.y - cc.y);
            const cplx yn = cmk(cc.x + (9.0 / 170.0) * ee.x, cc.y + (9.0 / 170.0) * ee.y);
            __stcs(a.sF + o, ee);
            a.sB[o] = yn;
        }
    } else {
#pragma unroll
        for (int k = 0; k < LISE_UPD_EPT; ++k) {
            const size_t el = e0 + (size_t)k * LISE_UPD_THREADS;
            if (el >= slen) continue;
            const size_t o = so + el;
            const cplx w = a.W[o];
            const cplx tt = (a.order == 1) ? a.sA[o] : a.sG[o];
            const cplx gg = cmk((w.y - eta * tt.y) * ih, -(w.x - eta * tt.x) * ih);
            const double cf = a.dt / (double)a.order;
            const cplx tn = cmk(cf * gg.x, cf * gg.y);
            a.sG[o] = tn;
            if (a.order == 1) { if (a.write_f) a.sC[o] = gg; a.sF[o] = cadd(tt, tn); }
            else a.sF[o] = cadd(a.sF[o], tn);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// density contributions of one axis (Eq. 3 with phi = conj(v), tau via Eq. 51) on a strip of 4 lines of the
// RAW v planes, accumulated into registers acc[m * NTH + r][3] (same thread <-> point map as taxis_core5):
//   WHICH = 0 (first derivative):  [0] += j_axis,  [1], [2] += the two J components
//             axis x: (+Xy -> J_z, -Xz -> J_y)   y: (+Xz -> J_x, -Xx -> J_z)   z: (+Xx -> J_y, -Xy -> J_x)
//   WHICH = 1 (second derivative): [0] += t = sum_s Re(phi_s^* D2 phi_s)
// ------------------------------------------------------------------------------------------------
template <int N, int AXIS, int WHICH>
__device__ __forceinline__ void dens_axis_task5(const cplx* __restrict__ v_u, const cplx* __restrict__ v_d,
                                                double (&acc)[TaskGeom<N>::NA][3], int l0, int LS, int PS,
                                                const double* __restrict__ tab)
{
    typedef LOp<N> L;
    constexpr int R = L::R, NTH = L::NTH, NKH = L::NKH, H = L::H;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const bool im = g & 1;
    const unsigned cs = im ? 0x80000000u : 0u;              // phi = conj(v)
    const int ibase = (l0 + (g >> 1)) * LS + t * PS;
    const int obase = (l0 + t) * LS + g * PS;
    Frags<N> F;
    F.load(tab, WHICH, g, t);
    double au[R][NTH][2], ad[R][NTH][2];
    zero_acc<N>(au); zero_acc<N>(ad);
#pragma unroll
    for (int kk = 0; kk < NKH; ++kk) {
        double xu[R], xd[R], vu[R], vd[R];
#pragma unroll
        for (int m = 0; m < R; ++m) {
            const int ii = ibase + (H * m + 4 * kk) * PS;
            xu[m] = xor_sign(ld_part(v_u, ii, im), cs); xd[m] = xor_sign(ld_part(v_d, ii, im), cs);
        }
        RDFT<R>::fwd(xu, vu); RDFT<R>::fwd(xd, vd);
        mma_blocks<N>(au, F, vu, kk); mma_blocks<N>(ad, F, vd, kk);
    }
    post_transform<N>(au); post_transform<N>(ad);
#pragma unroll
    for (int m = 0; m < R; ++m)
#pragma unroll
        for (int r = 0; r < NTH; ++r) {
            if (8 * r + g >= H) continue;
            const int idx = m * NTH + r;
            const int oi = obase + (H * m + 8 * r) * PS;
            const cplx fu = cconj(v_u[oi]), fd = cconj(v_d[oi]);
            const cplx du = cmk(au[m][r][0], au[m][r][1]), dd = cmk(ad[m][r][0], ad[m][r][1]);
            if (WHICH == 1) {
                acc[idx][0] += fu.x * du.x + fu.y * du.y + fd.x * dd.x + fd.y * dd.y;
            } else {
                const double ju = fu.x * du.y - fu.y * du.x, jd = fd.x * dd.y - fd.y * dd.x;
                // z1 = conj(phi_up) a_dn, z2 = conj(phi_dn) a_up
                const double z1r = fu.x * dd.x + fu.y * dd.y, z1i = fu.x * dd.y - fu.y * dd.x;
                const double z2r = fd.x * du.x + fd.y * du.y, z2i = fd.x * du.y - fd.y * du.x;
                const double Xx = z1i + z2i, Xy = -z1r + z2r, Xz = ju - jd;
                acc[idx][0] += ju + jd;
                if (AXIS == 0)      { acc[idx][1] += Xy; acc[idx][2] -= Xz; }
                else if (AXIS == 1) { acc[idx][1] += Xz; acc[idx][2] -= Xx; }
                else                { acc[idx][1] += Xx; acc[idx][2] -= Xy; }
            }
        }
}

// part[field][base + line * GLS + row * GPS] += acc of one task (the thread's own points)
template <int N, int AXIS>
__device__ __forceinline__ void dens_task_flush5(double* __restrict__ part, int nxyz, int which, const double (&acc)[TaskGeom<N>::NA][3],
                                                 int base, int l0, int GLS, int GPS)
{
    typedef LOp<N> L;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int f1 = (AXIS == 0) ? ACC_J + 2 : (AXIS == 1) ? ACC_J + 0 : ACC_J + 1;
    const int f2 = (AXIS == 0) ? ACC_J + 1 : (AXIS == 1) ? ACC_J + 2 : ACC_J + 0;
#pragma unroll
    for (int m = 0; m < L::R; ++m)
#pragma unroll
        for (int r = 0; r < L::NTH; ++r) {
            if (8 * r + g >= L::H) continue;
            const int idx = m * L::NTH + r, n = L::H * m + 8 * r + g;
            const size_t gi = (size_t)base + (size_t)(l0 + t) * GLS + (size_t)n * GPS;
            if (which == 1) part[(size_t)ACC_T * nxyz + gi] += acc[idx][0];
            else {
                part[(size_t)(ACC_JC + AXIS) * nxyz + gi] += acc[idx][0];
                part[(size_t)f1 * nxyz + gi] += acc[idx][1];
                part[(size_t)f2 * nxyz + gi] += acc[idx][2];
            }
        }
}

// ------------------------------------------------------------------------------------------------
// densities of the states in Z on yz-planes: pointwise n, s, kappa (Eq. 3a, 3d, 3b) and the y/z-line parts of
// t, j, J.  grid (nx, G), NWARP warps; v_up, v_dn planes prefetched by cp.async (two buffers), one barrier per state.
// Every accumulator lives in registers for the whole launch (fixed thread <-> point maps) and is added to part[g]
// at the end, map by map (deterministic).   shared: tables | v[2][SB][2][PP]
// ------------------------------------------------------------------------------------------------
template <int NY, int NZ, int NWARP, int SB>
__global__ void __maxnreg__(coresident_regs(NWARP)) k5_dens_yz(DArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int LD = ldpad(NZ), PP = NY * LD, NPTS = NY * NZ, NTHR = NWARP * 32;
    constexpr int NIT = (NPTS + NTHR - 1) / NTHR;
    constexpr int NTY = 2 * (NZ / 4), NTZ = 2 * (NY / 4), NTASK = NTY + NTZ, TPW = (NTASK + NWARP - 1) / NWARP;
    constexpr int NAY = TaskGeom<NY>::NA, NAZ = TaskGeom<NZ>::NA, NAM = NAY > NAZ ? NAY : NAZ;
    const int nxyz = a.L.nxyz;
    const int gbase = blockIdx.x * NPTS;
    double* s_ty = (double*)smem;
    double* s_tz = s_ty + LOp<NY>::TABSZ;
    cplx* vpl = (cplx*)(s_tz + LOp<NZ>::TABSZ + ((LOp<NY>::TABSZ + LOp<NZ>::TABSZ) & 1));   // [2][2][PP]
    for (int i = threadIdx.x; i < LOp<NY>::TABSZ; i += blockDim.x) s_ty[i] = a.stab[1][i];
    for (int i = threadIdx.x; i < LOp<NZ>::TABSZ; i += blockDim.x) s_tz[i] = a.stab[2][i];
    double accp[NIT][6];
    double acct[TPW][NAM][3];
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
        for (int k = 0; k < 6; ++k) accp[i][k] = 0.0;
#pragma unroll
    for (int i = 0; i < TPW; ++i)
#pragma unroll
        for (int r = 0; r < NAM; ++r) acct[i][r][0] = acct[i][r][1] = acct[i][r][2] = 0.0;
    const int warp = threadIdx.x >> 5;

    // a batch = SB states of this CTA's group (one barrier and one prefetch per batch, not per state)
    auto issue = [&](int st0, int buf) {
        for (int j = 0; j < SB; ++j) {
            const int st = st0 + j * a.G;
            if (st >= a.ns) break;
            const cplx* Zs = a.Z + ((size_t)st * 4 + 2) * nxyz + gbase;
            cplx* dst = vpl + (buf * SB + j) * 2 * PP;
            for (int i = threadIdx.x; i < 2 * NPTS; i += blockDim.x) {
                const int c = i / NPTS, p = i - c * NPTS, y = p / NZ, z = p - y * NZ;
                cp_async16(dst + c * PP + y * LD + z, Zs + (size_t)c * nxyz + p);
            }
        }
        cp_async_commit();
    };

    int st0 = blockIdx.y;
    if (st0 < a.ns) issue(st0, 0);
    for (int it = 0; st0 < a.ns; st0 += SB * a.G, ++it) {
        const int buf = it & 1;
        cp_async_wait<0>();
        __syncthreads();
        if (st0 + SB * a.G < a.ns) issue(st0 + SB * a.G, buf ^ 1);
        for (int j = 0; j < SB; ++j) {
        const int st = st0 + j * a.G;
        if (st >= a.ns) break;
        const cplx *vu_p = vpl + (buf * SB + j) * 2 * PP, *vd_p = vu_p + PP;
        // the up component of u for kappa: issued before the DMMA work, consumed after it
        cplx uu[NIT];
#pragma unroll
        for (int i = 0; i < NIT; ++i) {
            const int p = threadIdx.x + i * NTHR;
            uu[i] = (p < NPTS) ? a.Z[(size_t)st * 4 * nxyz + gbase + p] : cmk(0.0, 0.0);
        }
#pragma unroll
        for (int i = 0; i < TPW; ++i) {
            const int task = warp + i * NWARP;
            if (task < NTY) {
                const int l0 = 4 * (task >> 1);
                double (&ac)[NAY][3] = reinterpret_cast<double (&)[NAY][3]>(acct[i]);
                if (task & 1) dens_axis_task5<NY, 1, 1>(vu_p, vd_p, ac, l0, 1, LD, s_ty);
                else          dens_axis_task5<NY, 1, 0>(vu_p, vd_p, ac, l0, 1, LD, s_ty);
            } else if (task < NTASK) {
                const int tz = task - NTY, l0 = 4 * (tz >> 1);
                double (&ac)[NAZ][3] = reinterpret_cast<double (&)[NAZ][3]>(acct[i]);
                if (tz & 1) dens_axis_task5<NZ, 2, 1>(vu_p, vd_p, ac, l0, LD, 1, s_tz);
                else        dens_axis_task5<NZ, 2, 0>(vu_p, vd_p, ac, l0, LD, 1, s_tz);
            }
        }
        // pointwise densities: n (Eq. 3a), s = phi^+ sigma phi with phi = conj(v) (Eq. 3d), kappa (Eq. 3b)
#pragma unroll
        for (int i = 0; i < NIT; ++i) {
            const int p = threadIdx.x + i * NTHR;
            if (p >= NPTS) continue;
            const int y = p / NZ, z = p - y * NZ, si = y * LD + z;
            const cplx vu = vu_p[si], vd = vd_p[si], nu0 = uu[i];
            const double nu = vu.x * vu.x + vu.y * vu.y, nd = vd.x * vd.x + vd.y * vd.y;
            const double zr = vu.x * vd.x + vu.y * vd.y, zi = vu.y * vd.x - vu.x * vd.y;   // v_up conj(v_dn)
            accp[i][0] += nu + nd;
            accp[i][1] += 2.0 * zr;
            accp[i][2] += 2.0 * zi;
            accp[i][3] += nu - nd;
            accp[i][4] += vd.x * nu0.x + vd.y * nu0.y;      // conj(v_dn) u_up
            accp[i][5] += vd.x * nu0.y - vd.y * nu0.x;
        }
        }
    }
    double* part = a.part + (size_t)blockIdx.y * LISE_NACC * nxyz;
    const int prow[6] = {ACC_N, ACC_S + 0, ACC_S + 1, ACC_S + 2, ACC_K + 0, ACC_K + 1};
#pragma unroll
    for (int i = 0; i < NIT; ++i) {
        const int p = threadIdx.x + i * NTHR;
        if (p >= NPTS) continue;
#pragma unroll
        for (int k = 0; k < 6; ++k) part[(size_t)prow[k] * nxyz + gbase + p] += accp[i][k];
    }
    // the y-task and z-task maps touch the same fields (J components): one map at a time
#pragma unroll
    for (int i = 0; i < TPW; ++i) {
        const int task = warp + i * NWARP;
        if (task < NTY) {
            const double (&ac)[NAY][3] = reinterpret_cast<const double (&)[NAY][3]>(acct[i]);
            dens_task_flush5<NY, 1>(part, nxyz, task & 1, ac, gbase, 4 * (task >> 1), 1, NZ);
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < TPW; ++i) {
        const int task = warp + i * NWARP;
        if (task >= NTY && task < NTASK) {
            const int tz = task - NTY;
            const double (&ac)[NAZ][3] = reinterpret_cast<const double (&)[NAZ][3]>(acct[i]);
            dens_task_flush5<NZ, 2>(part, nxyz, tz & 1, ac, gbase, 4 * (tz >> 1), NZ, 1);
        }
    }
}

// x-axis density pass of the states in Z.   grid (ny, G), NWARP warps.  shared: table | v[2][2][PP]
template <int NX, int NZ, int NWARP, int SB>
__global__ void __maxnreg__(coresident_regs(NWARP)) k5_dens_x(DArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int LD = ldpad(NZ), PP = NX * LD, NPTS = NX * NZ;
    constexpr int NTX = 2 * (NZ / 4), TPW = (NTX + NWARP - 1) / NWARP;
    constexpr int NA = TaskGeom<NX>::NA;
    typedef LOp<NX> L;
    const int nxyz = a.L.nxyz, gs = a.L.ny * NZ, gb = blockIdx.x * NZ;
    double* s_tx = (double*)smem;
    cplx* vpl = (cplx*)(s_tx + L::TABSZ + (L::TABSZ & 1));
    for (int i = threadIdx.x; i < L::TABSZ; i += blockDim.x) s_tx[i] = a.stab[0][i];
    double acc[TPW][NA][3];
#pragma unroll
    for (int i = 0; i < TPW; ++i)
#pragma unroll
        for (int r = 0; r < NA; ++r) acc[i][r][0] = acc[i][r][1] = acc[i][r][2] = 0.0;
    const int warp = threadIdx.x >> 5;

    auto issue = [&](int st0, int buf) {
        for (int j = 0; j < SB; ++j) {
            const int st = st0 + j * a.G;
            if (st >= a.ns) break;
            const cplx* Zs = a.Z + ((size_t)st * 4 + 2) * nxyz + gb;
            cplx* dst = vpl + (buf * SB + j) * 2 * PP;
            for (int i = threadIdx.x; i < 2 * NPTS; i += blockDim.x) {
                const int c = i / NPTS, p = i - c * NPTS, x = p / NZ, z = p - x * NZ;
                cp_async16(dst + c * PP + x * LD + z, Zs + (size_t)c * nxyz + (size_t)x * gs + z);
            }
        }
        cp_async_commit();
    };

    int st0 = blockIdx.y;
    if (st0 < a.ns) issue(st0, 0);
    for (int it = 0; st0 < a.ns; st0 += SB * a.G, ++it) {
        const int buf = it & 1;
        cp_async_wait<0>();
        __syncthreads();
        if (st0 + SB * a.G < a.ns) issue(st0 + SB * a.G, buf ^ 1);
        for (int j = 0; j < SB; ++j) {
        if (st0 + j * a.G >= a.ns) break;
        const cplx *vu_p = vpl + (buf * SB + j) * 2 * PP, *vd_p = vu_p + PP;
#pragma unroll
        for (int i = 0; i < TPW; ++i) {
            const int task = warp + i * NWARP;
            if (task < NTX) {
                const int l0 = 4 * (task >> 1);
                if (task & 1) dens_axis_task5<NX, 0, 1>(vu_p, vd_p, acc[i], l0, 1, LD, s_tx);
                else          dens_axis_task5<NX, 0, 0>(vu_p, vd_p, acc[i], l0, 1, LD, s_tx);
            }
        }
        }
    }
    double* part = a.part + (size_t)blockIdx.y * LISE_NACC * nxyz;
#pragma unroll
    for (int i = 0; i < TPW; ++i) {
        const int task = warp + i * NWARP;
        if (task < NTX) dens_task_flush5<NX, 0>(part, nxyz, task & 1, acc[i], gb, 4 * (task >> 1), 1, gs);
    }
}
