// plane4_kernels.cuh -- the per-state kernels on the fp64 tensor-core path ("v4").
//
// Decomposition: h = V_loc + sum_i T_i, T_i acting on lattice lines along axis i;
// a CTA OWNS one lattice plane for the whole launch (grid = planes x G state groups <= SM count) and loops
// over work units (a unit = NCOMP components of one state on that plane).
//   * shared-memory planes are stored [n1][LD] with LD = n2 padded so that LD % 8 == 4 (in 16-byte units):
//     the 16 distinct operand addresses of a DMMA fragment load then fall into two conflict-free wavefronts;
//   * the potentials of the plane are staged once per launch in compact form (M, A_i, W/2);
//   * the next unit's wavefunction plane is prefetched with cp.async into a second buffer while the DMMA
//     passes of the current unit run (NBUF = 2), so global-memory latency is off the critical path;
//   * V_loc, the pairing block and -conj(.) for the v pair are folded into the store phase.
// Line operator: D_i, D2_i as circulant DMMA tiles (Eq. 48), mma.sync.m8n8k4.f64:
//   out[n][col] = sum_m c[n - m] x[m][col], A = circulant tile (row 8r+g, k 4k+t), B = x tile (k 4k+t,
//   column g = (line l0 + g/2, re|im)), accumulator row 8r+g, columns 2t, 2t+1 = (re, im) of line l0 + t.
// Requires every lattice edge to be a multiple of 4.
#pragma once
#include "common.cuh"
#include "state_kernels.cuh"

__host__ __device__ constexpr int ldpad(int n) { return n + ((4 - n % 8) + 8) % 8; }

__device__ __forceinline__ void dmma4(double (&d)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NPENDING) : "memory"); }

template <int N>
struct Line4 {
    static constexpr int NK = N / 4;                           // k steps
    static constexpr int NT = (N + 7) / 8;                     // output row tiles
    static constexpr int RT = (NT <= 5) ? NT : (NT + 1) / 2;   // row tiles per pass (bounds the accumulators)
};

// circulant fragments of this thread: cf[j] = c[(4j + g - t) mod N]   (ct: doubled table, ct[N + d])
template <int N>
__device__ __forceinline__ void load_cf4(const double2* __restrict__ ct, int g, int t, double (&cf1)[N / 4], double (&cf2)[N / 4])
{
#pragma unroll
    for (int j = 0; j < N / 4; ++j) {
        const int d = (4 * j + g - t + N) % N;
        const double2 c = ct[N + d];
        cf1[j] = c.x; cf2[j] = c.y;
    }
}

// compact potentials of one plane for one axis, in shared memory (doubles, same padded layout as the planes)
//   B_i = A_i + (sigma x W)_i / 2:  x: b00 = A - hWy, b11 = A + hWy, b01 = (0, -hWz)
//                                   y: b00 = A + hWx, b11 = A - hWx, b01 = (-hWz, 0)
//                                   z: b00 = b11 = A,               b01 = (hWy, hWx)        (hW = W / 2)
struct AxisPot4 {
    const double* M;      // hbar^2 / 2m*
    const double* A;      // A_axis
    const double* w1;     // x: hWy   y: hWx   z: hWy
    const double* w2;     // x: hWz   y: hWz   z: hWx
};

template <int AXIS>
__device__ __forceinline__ void make_B4(double A, double w1, double w2, double& b00, double& b11, double& br, double& bi)
{
    if (AXIS == 0)      { b00 = A - w1; b11 = A + w1; br = 0.0; bi = -w2; }
    else if (AXIS == 1) { b00 = A + w1; b11 = A - w1; br = -w2; bi = 0.0; }
    else                { b00 = A;      b11 = A;      br = w1;  bi = w2; }
}

// the part (re if !im, im if im) of g = -i B phi this lane feeds to the tensor core
template <int AXIS>
__device__ __forceinline__ void g_part4(bool im, double A, double w1, double w2, cplx fu, cplx fd, double& xgu, double& xgd)
{
    // T = B phi;  g = (T.im, -T.re):  lane value = im ? -T.re : T.im
    // "own" part p (re for im-lanes, im otherwise) and the other part o of each component
    const double pu = im ? fu.x : fu.y, pd = im ? fd.x : fd.y;
    const double ou = im ? fu.y : fu.x, od = im ? fd.y : fd.x;
    const double sg = im ? -1.0 : 1.0;
    double tu, td;
    if (AXIS == 0) {            // b01 = (0, beta), beta = -w2:  T_u.re = b00 ur - beta di, T_u.im = b00 ui + beta dr
        const double beta = -w2;                                 //   T_d.re = b11 dr + beta ui, T_d.im = b11 di - beta ur
        tu = (A - w1) * pu + (im ? -beta : beta) * od;
        td = (A + w1) * pd + (im ? beta : -beta) * ou;
    } else if (AXIS == 1) {     // b01 = (alpha, 0), alpha = -w2:  T_u = b00 phi_u + alpha phi_d, T_d = b11 phi_d + alpha phi_u
        tu = (A + w1) * pu - w2 * pd;
        td = (A - w1) * pd - w2 * pu;
    } else {                    // b01 = (alpha, beta) = (w1, w2):
        // T_u.re = A ur + alpha dr - beta di ; T_u.im = A ui + alpha di + beta dr
        // T_d.re = A dr + alpha ur + beta ui ; T_d.im = A di + alpha ui - beta ur
        tu = A * pu + w1 * pd + (im ? -w2 : w2) * od;
        td = A * pd + w1 * pu + (im ? w2 : -w2) * ou;
    }
    xgu = sg * tu; xgd = sg * td;
}

// T_i phi of one 2-spinor on a strip of 4 lines.  ACCUM 0: out = result, 1: out += result,
// 2: out += result mapped back to the raw v space, -conj(result) (out then holds W, not h phi).
// CONJ: the planes hold raw v components; phi = conj(v) is formed on the fly.
template <int N, int AXIS, int ACCUM, bool CONJ>
__device__ __forceinline__ void happly_axis_task4(const cplx* __restrict__ phi_u, const cplx* __restrict__ phi_d,
                                                  cplx* __restrict__ out_u, cplx* __restrict__ out_d,
                                                  const AxisPot4 pot, int l0, int LS, int PS, const double2* __restrict__ ct)
{
    typedef Line4<N> T;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    double cf1[T::NK], cf2[T::NK];
    load_cf4<N>(ct, g, t, cf1, cf2);
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
            cplx fu = phi_u[ii], fd = phi_d[ii];
            if (CONJ) { fu.y = -fu.y; fd.y = -fd.y; }
            const double M = pot.M[ii], A = pot.A[ii], w1 = pot.w1[ii], w2 = pot.w2[ii];
            double xgu, xgd;
            g_part4<AXIS>(im, A, w1, w2, fu, fd, xgu, xgd);                   // g = -i B phi
            const double xfu = im ? fu.y : fu.x, xfd = im ? fd.y : fd.x;
            const double mh = -0.5 * M;
            const double xqu = mh * xfu, xqd = mh * xfd;                      // q = -M phi / 2
#pragma unroll
            for (int r = 0; r < T::RT; ++r) {
                if (r0 + r >= T::NT) continue;
                const int j = (((2 * (r0 + r) - k) % T::NK) + T::NK) % T::NK;
                dmma4(au[r], cf1[j], xfu); dmma4(ad[r], cf1[j], xfd);
                dmma4(bu[r], cf2[j], xfu); dmma4(bd[r], cf2[j], xfd);
                dmma4(cu[r], cf1[j], xgu); dmma4(cd[r], cf1[j], xgd);
                dmma4(cu[r], cf2[j], xqu); dmma4(cd[r], cf2[j], xqd);
            }
        }
#pragma unroll
        for (int r = 0; r < T::RT; ++r) {
            if (r0 + r >= T::NT) continue;
            if (8 * (r0 + r) + g >= N) continue;                              // padding rows
            const int oi = obase + 8 * (r0 + r) * PS;
            const double M = pot.M[oi];
            double b00, b11, br, bi;
            make_B4<AXIS>(pot.A[oi], pot.w1[oi], pot.w2[oi], b00, b11, br, bi);
            cplx lu, ld_;
            apply_C(b00, b11, cmk(br, bi), cmk(au[r][0], au[r][1]), cmk(ad[r][0], ad[r][1]), lu, ld_);   // -i B D phi
            cplx ru = cmk(lu.x - 0.5 * M * bu[r][0] + cu[r][0], lu.y - 0.5 * M * bu[r][1] + cu[r][1]);
            cplx rd = cmk(ld_.x - 0.5 * M * bd[r][0] + cd[r][0], ld_.y - 0.5 * M * bd[r][1] + cd[r][1]);
            if (ACCUM == 1) { const cplx ou = out_u[oi], od = out_d[oi]; ru = cadd(ru, ou); rd = cadd(rd, od); }
            if (ACCUM == 2) {
                const cplx ou = out_u[oi], od = out_d[oi];
                ru = cmk(ou.x - ru.x, ou.y + ru.y); rd = cmk(od.x - rd.x, od.y + rd.y);
            }
            out_u[oi] = ru; out_d[oi] = rd;
        }
    }
}

// rows of the V_loc / pairing staging area pV (VSTAGE) and their source rows in the potential array
__device__ __forceinline__ void load_vloc(const double* __restrict__ pot, int nxyz, int gi, double (&v)[6])
{
    v[0] = pot[(size_t)P_ULOC * nxyz + gi];
    v[1] = pot[(size_t)(P_S + 0) * nxyz + gi]; v[2] = pot[(size_t)(P_S + 1) * nxyz + gi]; v[3] = pot[(size_t)(P_S + 2) * nxyz + gi];
    v[4] = pot[(size_t)P_DELTA * nxyz + gi];   v[5] = pot[(size_t)(P_DELTA + 1) * nxyz + gi];
}

// ------------------------------------------------------------------------------------------------
// H-apply, yz-planes:  W = [V_loc + T_y + T_z] X + pairing block (Eq. 11, mu = 0).
// grid (nx, G), NWARP warps.  A unit = NCOMP components (NCOMP = 4: a state, 2: one 2-spinor) on the plane.
// shared: tables | phi[NBUF][NCOMP][PP] | out[NCOMP][PP] | pots M, Ay, Az, hWx, hWy, hWz [PP] | pV[6][PP] (VSTAGE)
// ------------------------------------------------------------------------------------------------
template <int NY, int NZ, int NCOMP, int NBUF, int NWARP, bool VSTAGE>
__global__ void __launch_bounds__(NWARP * 32, 1) k4_happly_yz(HArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int LD = ldpad(NZ), PP = NY * LD, NPTS = NY * NZ;
    constexpr int NPAIR = NCOMP / 2, UPS = 4 / NCOMP;
    const int nxyz = a.L.nxyz;
    const int gbase = blockIdx.x * NPTS;
    double2* s_cty = smem;
    double2* s_ctz = s_cty + 2 * NY;
    cplx* phi = s_ctz + 2 * NZ;
    cplx* out = phi + NBUF * NCOMP * PP;
    double* pM = (double*)(out + NCOMP * PP);
    double *pAy = pM + PP, *pAz = pAy + PP, *pWx = pAz + PP, *pWy = pWx + PP, *pWz = pWy + PP;
    double* pV = pWz + PP;
    const double* pot = a.pot;
    stage_table(s_cty, a.ctab[1], NY);
    stage_table(s_ctz, a.ctab[2], NZ);
    for (int p = threadIdx.x; p < NPTS; p += blockDim.x) {
        const int y = p / NZ, z = p - y * NZ, si = y * LD + z, gi = gbase + p;
        pM[si] = pot[(size_t)P_M * nxyz + gi];
        pAy[si] = pot[(size_t)(P_A + 1) * nxyz + gi]; pAz[si] = pot[(size_t)(P_A + 2) * nxyz + gi];
        pWx[si] = 0.5 * pot[(size_t)(P_W + 0) * nxyz + gi]; pWy[si] = 0.5 * pot[(size_t)(P_W + 1) * nxyz + gi];
        pWz[si] = 0.5 * pot[(size_t)(P_W + 2) * nxyz + gi];
        if (VSTAGE) {
            double v[6]; load_vloc(pot, nxyz, gi, v);
#pragma unroll
            for (int k = 0; k < 6; ++k) pV[k * PP + si] = v[k];
        }
    }
    const AxisPot4 poty = {pM, pAy, pWx, pWz}, potz = {pM, pAz, pWy, pWx};
    const int warp = threadIdx.x >> 5;
    const int nunits = a.ns * UPS;

    auto issue = [&](int u, int buf) {
        const int st = u / UPS, pg = u - st * UPS;
        const cplx* Xs = a.X + ((size_t)st * 4 + pg * NCOMP) * nxyz + gbase;
        cplx* dst = phi + buf * NCOMP * PP;
        for (int i = threadIdx.x; i < NCOMP * NPTS; i += blockDim.x) {
            const int c = i / NPTS, p = i - c * NPTS, y = p / NZ, z = p - y * NZ;
            cp_async16(dst + c * PP + y * LD + z, Xs + (size_t)c * nxyz + p);
        }
        cp_async_commit();
    };

    int u = blockIdx.y;
    if (u < nunits) issue(u, 0);
    for (int it = 0; u < nunits; u += a.G, ++it) {
        const int buf = (NBUF == 2) ? (it & 1) : 0;
        if (NBUF == 2 && u + a.G < nunits) { issue(u + a.G, buf ^ 1); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const int st = u / UPS, pg = u - st * UPS;
        cplx* phib = phi + buf * NCOMP * PP;
        // ---- y lines (one per z): LS = 1, PS = LD ----
        for (int task = warp; task < NPAIR * (NZ / 4); task += NWARP) {
            const int pr = task / (NZ / 4), l0 = 4 * (task - pr * (NZ / 4));
            const cplx *fu = phib + 2 * pr * PP, *fd = fu + PP;
            cplx *ou = out + 2 * pr * PP, *od = ou + PP;
            if (pg * NPAIR + pr) happly_axis_task4<NY, 1, 0, true>(fu, fd, ou, od, poty, l0, 1, LD, s_cty);
            else                 happly_axis_task4<NY, 1, 0, false>(fu, fd, ou, od, poty, l0, 1, LD, s_cty);
        }
        __syncthreads();
        // ---- z lines (one per y): LS = LD, PS = 1 ----
        for (int task = warp; task < NPAIR * (NY / 4); task += NWARP) {
            const int pr = task / (NY / 4), l0 = 4 * (task - pr * (NY / 4));
            const cplx *fu = phib + 2 * pr * PP, *fd = fu + PP;
            cplx *ou = out + 2 * pr * PP, *od = ou + PP;
            if (pg * NPAIR + pr) happly_axis_task4<NZ, 2, 1, true>(fu, fd, ou, od, potz, l0, LD, 1, s_ctz);
            else                 happly_axis_task4<NZ, 2, 1, false>(fu, fd, ou, od, potz, l0, LD, 1, s_ctz);
        }
        __syncthreads();
        // ---- V_loc, pairing block, -conj(.) for the v pair; store ----
        const cplx* Xst = a.X + (size_t)st * 4 * nxyz;
        cplx* Ws = a.W + (size_t)st * 4 * nxyz;
        for (int p = threadIdx.x; p < NPTS; p += blockDim.x) {
            const int y = p / NZ, z = p - y * NZ, si = y * LD + z, gi = gbase + p;
            double v[6];
            if (VSTAGE) {
#pragma unroll
                for (int k = 0; k < 6; ++k) v[k] = pV[k * PP + si];
            } else load_vloc(pot, nxyz, gi, v);
            const double ul = v[0], sx = v[1], sy = v[2], sz = v[3];
            const cplx Dl = cmk(v[4], v[5]);
#pragma unroll
            for (int pr = 0; pr < NPAIR; ++pr) {
                const int pair = pg * NPAIR + pr;
                cplx fu = phib[(2 * pr) * PP + si], fd = phib[(2 * pr + 1) * PP + si];
                if (pair) { fu = cconj(fu); fd = cconj(fd); }
                cplx ou = out[(2 * pr) * PP + si], od = out[(2 * pr + 1) * PP + si];
                caxpy(ou, ul + sz, fu); cfma(ou, cmk(sx, -sy), fd);
                caxpy(od, ul - sz, fd); cfma(od, cmk(sx, sy), fu);
                if (pair == 0) {
                    cplx vu, vd;
                    if (NCOMP == 4) { vu = phib[2 * PP + si]; vd = phib[3 * PP + si]; }
                    else { vu = Xst[(size_t)2 * nxyz + gi]; vd = Xst[(size_t)3 * nxyz + gi]; }
                    cfma(ou, Dl, vd);
                    cfma(od, cmk(-Dl.x, -Dl.y), vu);
                } else {
                    cplx uu, ud;
                    if (NCOMP == 4) { uu = phib[si]; ud = phib[PP + si]; }
                    else { uu = Xst[gi]; ud = Xst[(size_t)nxyz + gi]; }
                    const cplx Dc = cconj(Dl);
                    ou = cmk(-ou.x, ou.y); od = cmk(-od.x, od.y);           // -conj(h conj v)
                    cfma(ou, cmk(-Dc.x, -Dc.y), ud);
                    cfma(od, Dc, uu);
                }
                Ws[(size_t)(2 * pair) * nxyz + gi] = ou; Ws[(size_t)(2 * pair + 1) * nxyz + gi] = od;
            }
        }
        __syncthreads();
        if (NBUF == 1 && u + a.G < nunits) issue(u + a.G, 0);
    }
}

// ------------------------------------------------------------------------------------------------
// H-apply, xz-planes:  W += T_x X,  eta_part[st][pg * ny + iy] = dV Re <X|W> over the plane.
// grid (ny, G), NWARP warps.  The unit's X plane and its W plane (from k4_happly_yz) are both prefetched
// with cp.async; the x pass accumulates into the W plane in shared memory, which is then stored.
// shared: table | phi[NBUF][NCOMP][PP] | out[NBUF][NCOMP][PP] | pots M, Ax, hWy, hWz [PP] | red
// ------------------------------------------------------------------------------------------------
template <int NX, int NZ, int NCOMP, int NBUF, int NWARP>
__global__ void __launch_bounds__(NWARP * 32, 1) k4_happly_xz(HArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int LD = ldpad(NZ), PP = NX * LD, NPTS = NX * NZ;
    constexpr int NPAIR = NCOMP / 2, UPS = 4 / NCOMP;
    const int nxyz = a.L.nxyz, gs = a.L.ny * NZ, gb = blockIdx.x * NZ;
    double2* s_ctx = smem;
    cplx* phi = s_ctx + 2 * NX;
    cplx* out = phi + NBUF * NCOMP * PP;
    double* pM = (double*)(out + NBUF * NCOMP * PP);
    double *pAx = pM + PP, *pWy = pAx + PP, *pWz = pWy + PP;
    double* s_red = pWz + PP;
    const double* pot = a.pot;
    stage_table(s_ctx, a.ctab[0], NX);
    for (int p = threadIdx.x; p < NPTS; p += blockDim.x) {
        const int x = p / NZ, z = p - x * NZ, si = x * LD + z, gi = gb + x * gs + z;
        pM[si] = pot[(size_t)P_M * nxyz + gi];
        pAx[si] = pot[(size_t)(P_A + 0) * nxyz + gi];
        pWy[si] = 0.5 * pot[(size_t)(P_W + 1) * nxyz + gi]; pWz[si] = 0.5 * pot[(size_t)(P_W + 2) * nxyz + gi];
    }
    const AxisPot4 potx = {pM, pAx, pWy, pWz};
    const int warp = threadIdx.x >> 5;
    const int nunits = a.ns * UPS;

    auto issue = [&](int u, int buf) {
        const int st = u / UPS, pg = u - st * UPS;
        const size_t go = ((size_t)st * 4 + pg * NCOMP) * nxyz + gb;
        cplx* dphi = phi + buf * NCOMP * PP;
        cplx* dout = out + buf * NCOMP * PP;
        for (int i = threadIdx.x; i < NCOMP * NPTS; i += blockDim.x) {
            const int c = i / NPTS, p = i - c * NPTS, x = p / NZ, z = p - x * NZ;
            const size_t g = go + (size_t)c * nxyz + (size_t)x * gs + z;
            cp_async16(dphi + c * PP + x * LD + z, a.X + g);
            cp_async16(dout + c * PP + x * LD + z, a.W + g);
        }
        cp_async_commit();
    };

    int u = blockIdx.y;
    if (u < nunits) issue(u, 0);
    for (int it = 0; u < nunits; u += a.G, ++it) {
        const int buf = (NBUF == 2) ? (it & 1) : 0;
        if (NBUF == 2 && u + a.G < nunits) { issue(u + a.G, buf ^ 1); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const int st = u / UPS, pg = u - st * UPS;
        cplx* phib = phi + buf * NCOMP * PP;
        cplx* outb = out + buf * NCOMP * PP;
        // ---- x lines (one per z): LS = 1, PS = LD ----
        for (int task = warp; task < NPAIR * (NZ / 4); task += NWARP) {
            const int pr = task / (NZ / 4), l0 = 4 * (task - pr * (NZ / 4));
            const cplx *fu = phib + 2 * pr * PP, *fd = fu + PP;
            cplx *ou = outb + 2 * pr * PP, *od = ou + PP;
            if (pg * NPAIR + pr) happly_axis_task4<NX, 0, 2, true>(fu, fd, ou, od, potx, l0, 1, LD, s_ctx);
            else                 happly_axis_task4<NX, 0, 1, false>(fu, fd, ou, od, potx, l0, 1, LD, s_ctx);
        }
        __syncthreads();
        // ---- store W, eta partial ----
        double eta_loc = 0.0;
        cplx* Wg = a.W + ((size_t)st * 4 + pg * NCOMP) * nxyz + gb;
        for (int i = threadIdx.x; i < NCOMP * NPTS; i += blockDim.x) {
            const int c = i / NPTS, p = i - c * NPTS, x = p / NZ, z = p - x * NZ, si = c * PP + x * LD + z;
            const cplx w = outb[si], f = phib[si];
            Wg[(size_t)c * nxyz + (size_t)x * gs + z] = w;
            eta_loc += f.x * w.x + f.y * w.y;
        }
        const double tsum = block_sum(eta_loc, s_red);     // two __syncthreads inside: phib / outb are free afterwards
        if (threadIdx.x == 0) a.eta_part[((size_t)st * UPS + pg) * a.L.ny + blockIdx.x] = tsum * a.L.dV;
        __syncthreads();
        if (NBUF == 1 && u + a.G < nunits) issue(u + a.G, 0);
    }
}

// ------------------------------------------------------------------------------------------------
// density contributions of one axis (Eq. 3 with phi = conj(v), tau via Eq. 51) on a strip of 4 lines,
// accumulated into REGISTERS: a warp always works on the same strips, so each thread owns the same output
// points (row 8r+g of line l0+t) for every state of the launch.
//   WHICH = 0 (first derivative):  acc[r][0] += j_axis,  acc[r][1], acc[r][2] += the two J components
//             axis x: (+Xy -> J_z, -Xz -> J_y)   y: (+Xz -> J_x, -Xx -> J_z)   z: (+Xx -> J_y, -Xy -> J_x)
//   WHICH = 1 (second derivative): acc[r][0] += t = sum_s Re(phi_s^* D2 phi_s)
// ------------------------------------------------------------------------------------------------
template <int N, int AXIS, int WHICH>
__device__ __forceinline__ void dens_axis_task4(const cplx* __restrict__ phi_u, const cplx* __restrict__ phi_d,
                                                double (&acc)[(N + 7) / 8][3], int l0, int LS, int PS,
                                                const double2* __restrict__ ct)
{
    typedef Line4<N> T;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    double cf[T::NK];
#pragma unroll
    for (int j = 0; j < T::NK; ++j) {
        const double2 c = ct[N + (4 * j + g - t + N) % N];
        cf[j] = (WHICH == 0) ? c.x : c.y;
    }
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
                dmma4(au[r], cf[j], xfu); dmma4(ad[r], cf[j], xfd);
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
                acc[r0 + r][0] += fu.x * du.x + fu.y * du.y + fd.x * dd.x + fd.y * dd.y;
            } else {
                const double ju = fu.x * du.y - fu.y * du.x, jd = fd.x * dd.y - fd.y * dd.x;
                // z1 = conj(phi_up) a_dn, z2 = conj(phi_dn) a_up
                const double z1r = fu.x * dd.x + fu.y * dd.y, z1i = fu.x * dd.y - fu.y * dd.x;
                const double z2r = fd.x * du.x + fd.y * du.y, z2i = fd.x * du.y - fd.y * du.x;
                const double Xx = z1i + z2i, Xy = -z1r + z2r, Xz = ju - jd;
                acc[r0 + r][0] += ju + jd;
                if (AXIS == 0)      { acc[r0 + r][1] += Xy; acc[r0 + r][2] -= Xz; }
                else if (AXIS == 1) { acc[r0 + r][1] += Xz; acc[r0 + r][2] -= Xx; }
                else                { acc[r0 + r][1] += Xx; acc[r0 + r][2] -= Xy; }
            }
        }
    }
}

// part[field][base + line * GLS + row * GPS] += acc of one task (the thread's own points)
template <int N, int AXIS>
__device__ __forceinline__ void dens_task_flush(double* __restrict__ part, int nxyz, int which, const double (&acc)[(N + 7) / 8][3],
                                                int base, int l0, int GLS, int GPS)
{
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    // accumulator rows of the three slots of a first-derivative task
    const int f1 = (AXIS == 0) ? ACC_J + 2 : (AXIS == 1) ? ACC_J + 0 : ACC_J + 1;
    const int f2 = (AXIS == 0) ? ACC_J + 1 : (AXIS == 1) ? ACC_J + 2 : ACC_J + 0;
#pragma unroll
    for (int r = 0; r < (N + 7) / 8; ++r) {
        const int n = 8 * r + g;
        if (n >= N) continue;
        const size_t gi = (size_t)base + (size_t)(l0 + t) * GLS + (size_t)n * GPS;
        if (which == 1) part[(size_t)ACC_T * nxyz + gi] += acc[r][0];
        else {
            part[(size_t)(ACC_JC + AXIS) * nxyz + gi] += acc[r][0];
            part[(size_t)f1 * nxyz + gi] += acc[r][1];
            part[(size_t)f2 * nxyz + gi] += acc[r][2];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// ABM update fused with the pointwise and y/z-line density passes of the NEW state (modes as k_update_yz in
// state_kernels.cuh).  grid (nx, G), NWARP warps.   shared: tables | phi[2][PP]
// Every density accumulator of the plane lives in registers for the whole launch (fixed thread <-> point maps:
// pointwise map, y-task map, z-task map) and is added to part[g] once at the end, map by map (deterministic).
// ------------------------------------------------------------------------------------------------
template <int MODE, int NY, int NZ, int NWARP>
__global__ void __launch_bounds__(NWARP * 32, 1) k4_update_yz(UArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int LD = ldpad(NZ), PP = NY * LD, NPTS = NY * NZ, NTHR = NWARP * 32;
    constexpr int NIT = (NPTS + NTHR - 1) / NTHR;
    constexpr int NTY = 2 * (NZ / 4), TPWY = (NTY + NWARP - 1) / NWARP;
    constexpr int NTZ = 2 * (NY / 4), TPWZ = (NTZ + NWARP - 1) / NWARP;
    const int nxyz = a.L.nxyz;
    const int gbase = blockIdx.x * NPTS;
    double2* s_cty = smem;
    double2* s_ctz = s_cty + 2 * NY;
    cplx* phi = s_ctz + 2 * NZ;                       // [2][PP]
    double accp[NIT][6];
    double accy[TPWY][(NY + 7) / 8][3], accz[TPWZ][(NZ + 7) / 8][3];
    if (MODE != 3) {
        stage_table(s_cty, a.ctab[1], NY); stage_table(s_ctz, a.ctab[2], NZ);
#pragma unroll
        for (int i = 0; i < NIT; ++i)
#pragma unroll
            for (int k = 0; k < 6; ++k) accp[i][k] = 0.0;
#pragma unroll
        for (int i = 0; i < TPWY; ++i)
#pragma unroll
            for (int r = 0; r < (NY + 7) / 8; ++r) accy[i][r][0] = accy[i][r][1] = accy[i][r][2] = 0.0;
#pragma unroll
        for (int i = 0; i < TPWZ; ++i)
#pragma unroll
            for (int r = 0; r < (NZ + 7) / 8; ++r) accz[i][r][0] = accz[i][r][1] = accz[i][r][2] = 0.0;
        __syncthreads();
    }
    const int warp = threadIdx.x >> 5;
    const double ih = 1.0 / a.hbarc;
    const double c48 = a.dt / 48.0;

    for (int st = blockIdx.y; st < a.ns; st += a.G) {
        const size_t so = (size_t)st * 4 * nxyz;
        double eta = 0.0;
        if (MODE != 0) {
            if (MODE == 3 && a.order > 1) eta = a.eta_fix[st];
            else {
                for (int j = 0; j < a.neta; ++j) eta += a.eta_part[(size_t)st * a.neta + j];   // fixed order
                if (!a.remove_phase) eta = 0.0;
                if (MODE == 3 && blockIdx.x == 0 && threadIdx.x == 0) a.eta_fix[st] = eta;
            }
        }
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int p = threadIdx.x + it * NTHR;
            if (p >= NPTS) continue;
            const int gi = gbase + p;
            cplx nw[4];
#pragma unroll
            for (int h = 0; h < 2; ++h) {              // components in pairs: all loads of a pair in flight together
                const size_t o0 = so + (size_t)(2 * h) * nxyz + gi, o1 = o0 + nxyz;
                if (MODE == 0) {
                    nw[2 * h] = a.Z[o0]; nw[2 * h + 1] = a.Z[o1];
                } else if (MODE == 1) {
                    cplx w[2], y[2], ym[2], f1[2], f2[2], f3[2], e[2];
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const size_t o = c ? o1 : o0;
                        w[c] = a.W[o]; y[c] = a.sA[o]; ym[c] = a.sB[o]; f1[c] = a.sD[o]; f2[c] = a.sE[o]; f3[c] = a.sC[o]; e[c] = a.sF[o];
                    }
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const size_t o = c ? o1 : o0;
                        const cplx fn = cmk((w[c].y - eta * y[c].y) * ih, -(w[c].x - eta * y[c].x) * ih);
                        const cplx half = cmk(0.5 * (y[c].x + ym[c].x), 0.5 * (y[c].y + ym[c].y));
                        cplx pp, qq;
                        pp.x = half.x + c48 * (119.0 * fn.x - 99.0 * f1[c].x + 69.0 * f2[c].x - 17.0 * f3[c].x);
                        pp.y = half.y + c48 * (119.0 * fn.y - 99.0 * f1[c].y + 69.0 * f2[c].y - 17.0 * f3[c].y);
                        qq.x = half.x + c48 * (51.0 * fn.x + 3.0 * f1[c].x + f2[c].x);
                        qq.y = half.y + c48 * (51.0 * fn.y + 3.0 * f1[c].y + f2[c].y);
                        const cplx m = cmk(pp.x - (161.0 / 170.0) * e[c].x, pp.y - (161.0 / 170.0) * e[c].y);
                        a.sC[o] = fn; a.sF[o] = m; a.sG[o] = pp; a.sB[o] = qq;
                        nw[2 * h + c] = m;
                    }
                } else if (MODE == 2) {
                    cplx w[2], m[2], qq[2], pp[2];
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const size_t o = c ? o1 : o0;
                        w[c] = a.W[o]; m[c] = a.sF[o]; qq[c] = a.sB[o]; pp[c] = a.sG[o];
                    }
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const size_t o = c ? o1 : o0;
                        const cplx fm = cmk((w[c].y - eta * m[c].y) * ih, -(w[c].x - eta * m[c].x) * ih);
                        const cplx cc = cmk(qq[c].x + c48 * 17.0 * fm.x, qq[c].y + c48 * 17.0 * fm.y);
                        const cplx ee = cmk(pp[c].x - cc.x, pp[c].y - cc.y);
                        const cplx yn = cmk(cc.x + (9.0 / 170.0) * ee.x, cc.y + (9.0 / 170.0) * ee.y);
                        a.sB[o] = yn; a.sF[o] = ee;
                        nw[2 * h + c] = yn;
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const size_t o = c ? o1 : o0;
                        const cplx w = a.W[o];
                        const cplx tt = (a.order == 1) ? a.sA[o] : a.sG[o];
                        const cplx gg = cmk((w.y - eta * tt.y) * ih, -(w.x - eta * tt.x) * ih);
                        const double cf = a.dt / (double)a.order;
                        const cplx tn = cmk(cf * gg.x, cf * gg.y);
                        a.sG[o] = tn;
                        if (a.order == 1) { if (a.write_f) a.sC[o] = gg; a.sF[o] = cadd(tt, tn); }
                        else a.sF[o] = cadd(a.sF[o], tn);
                        nw[2 * h + c] = tn;
                    }
                }
            }
            if (MODE != 3) {
                // pointwise densities: n (Eq. 3a), s = phi^+ sigma phi with phi = conj(v) (Eq. 3d), kappa (Eq. 3b)
                const cplx nu0 = nw[0], vu = nw[2], vd = nw[3];
                const double nu = vu.x * vu.x + vu.y * vu.y, nd = vd.x * vd.x + vd.y * vd.y;
                const double zr = vu.x * vd.x + vu.y * vd.y, zi = vu.y * vd.x - vu.x * vd.y;   // v_up conj(v_dn)
                accp[it][0] += nu + nd;
                accp[it][1] += 2.0 * zr;
                accp[it][2] += 2.0 * zi;
                accp[it][3] += nu - nd;
                accp[it][4] += vd.x * nu0.x + vd.y * nu0.y;      // conj(v_dn) u_up
                accp[it][5] += vd.x * nu0.y - vd.y * nu0.x;
                const int y = p / NZ, z = p - y * NZ, si = y * LD + z;
                phi[si] = cconj(vu); phi[PP + si] = cconj(vd);
            }
        }
        if (MODE != 3) {
            __syncthreads();
            // y lines: LS = 1, PS = LD; tasks = strips x {first-derivative, second-derivative}
#pragma unroll
            for (int i = 0; i < TPWY; ++i) {
                const int task = warp + i * NWARP;
                if (task < NTY) {
                    const int l0 = 4 * (task >> 1);
                    if (task & 1) dens_axis_task4<NY, 1, 1>(phi, phi + PP, accy[i], l0, 1, LD, s_cty);
                    else          dens_axis_task4<NY, 1, 0>(phi, phi + PP, accy[i], l0, 1, LD, s_cty);
                }
            }
            // z lines: LS = LD, PS = 1 (reads only; no barrier needed between the two passes)
#pragma unroll
            for (int i = 0; i < TPWZ; ++i) {
                const int task = warp + i * NWARP;
                if (task < NTZ) {
                    const int l0 = 4 * (task >> 1);
                    if (task & 1) dens_axis_task4<NZ, 2, 1>(phi, phi + PP, accz[i], l0, LD, 1, s_ctz);
                    else          dens_axis_task4<NZ, 2, 0>(phi, phi + PP, accz[i], l0, LD, 1, s_ctz);
                }
            }
            __syncthreads();
        }
    }
    if (MODE != 3) {
        double* part = a.part + (size_t)blockIdx.y * LISE_NACC * nxyz;
        const int prow[6] = {ACC_N, ACC_S + 0, ACC_S + 1, ACC_S + 2, ACC_K + 0, ACC_K + 1};
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int p = threadIdx.x + it * NTHR;
            if (p >= NPTS) continue;
#pragma unroll
            for (int k = 0; k < 6; ++k) part[(size_t)prow[k] * nxyz + gbase + p] += accp[it][k];
        }
#pragma unroll
        for (int i = 0; i < TPWY; ++i) {
            const int task = warp + i * NWARP;
            if (task < NTY) dens_task_flush<NY, 1>(part, nxyz, task & 1, accy[i], gbase, 4 * (task >> 1), 1, NZ);
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < TPWZ; ++i) {
            const int task = warp + i * NWARP;
            if (task < NTZ) dens_task_flush<NZ, 2>(part, nxyz, task & 1, accz[i], gbase, 4 * (task >> 1), NZ, 1);
        }
    }
}

// x-axis density pass of the states in Z.   grid (ny, G), NWARP warps.  shared: table | phi[2][PP]
template <int NX, int NZ, int NWARP>
__global__ void __launch_bounds__(NWARP * 32, 1) k4_dens_x(DArgs a)
{
    extern __shared__ double2 smem[];
    constexpr int LD = ldpad(NZ), PP = NX * LD, NPTS = NX * NZ;
    constexpr int NTX = 2 * (NZ / 4), TPW = (NTX + NWARP - 1) / NWARP;
    const int nxyz = a.L.nxyz, gs = a.L.ny * NZ, gb = blockIdx.x * NZ;
    double2* s_ctx = smem;
    cplx* phi = s_ctx + 2 * NX;
    double acc[TPW][(NX + 7) / 8][3];
#pragma unroll
    for (int i = 0; i < TPW; ++i)
#pragma unroll
        for (int r = 0; r < (NX + 7) / 8; ++r) acc[i][r][0] = acc[i][r][1] = acc[i][r][2] = 0.0;
    stage_table(s_ctx, a.ctab[0], NX);
    const int warp = threadIdx.x >> 5;
    for (int st = blockIdx.y; st < a.ns; st += a.G) {
        const cplx* Zs = a.Z + (size_t)st * 4 * nxyz;
        __syncthreads();
        for (int p = threadIdx.x; p < NPTS; p += blockDim.x) {
            const int x = p / NZ, z = p - x * NZ, si = x * LD + z, gi = gb + x * gs + z;
            phi[si] = cconj(Zs[(size_t)2 * nxyz + gi]); phi[PP + si] = cconj(Zs[(size_t)3 * nxyz + gi]);
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < TPW; ++i) {
            const int task = warp + i * NWARP;
            if (task < NTX) {
                const int l0 = 4 * (task >> 1);
                if (task & 1) dens_axis_task4<NX, 0, 1>(phi, phi + PP, acc[i], l0, 1, LD, s_ctx);
                else          dens_axis_task4<NX, 0, 0>(phi, phi + PP, acc[i], l0, 1, LD, s_ctx);
            }
        }
    }
    double* part = a.part + (size_t)blockIdx.y * LISE_NACC * nxyz;
#pragma unroll
    for (int i = 0; i < TPW; ++i) {
        const int task = warp + i * NWARP;
        if (task < NTX) dens_task_flush<NX, 0>(part, nxyz, task & 1, acc[i], gb, 4 * (task >> 1), 1, gs);
    }
}
