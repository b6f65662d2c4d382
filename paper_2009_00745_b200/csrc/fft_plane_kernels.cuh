// fft_plane_kernels.cuh -- H-apply kernels with the FFT-cost line operator.
//
//   k6_happly_yz : W  = [V_loc + T_y + T_z] X (+ pairing block, PAIRING) (yz-plane owner CTAs)
//   k6_happly_xz : W += T_x X (+ pairing block), eta partial sums         (xz-plane owner CTAs; the pairing block is added
//                  here on lattices whose yz-plane units are 2-spinors, where the yz kernel cannot add it: 32^3)
//
// Decomposition: h = V_loc + sum_i T_i,
//   T_i phi = -(1/2) [ M D2_i phi + D2_i (M phi) ] - i [ B_i D_i phi + D_i (B_i phi) ],  B_i = A_i + (sigma x W)_i / 2.
// D_i and D2_i are REAL operators (Eqs. 49-50), so the real and the imaginary part of a component are
// independent real lines.  One THREAD owns one real line in registers and runs the generated straight-line
// real-input FFT codelets of line_codelets.cuh (inner: a = D x, b = D2 x; outer: c = D g + D2 q): no data exchange
// inside a transform.  The only exchange is pointwise: B couples the two spin components and -i couples re and im,
// so the four lanes that hold (spin, part) of the same line -- lane = 8 * (2 * spin + part) + line -- swap their
// values of a by warp shuffles.  Between the two codelets the first half of the result (r1) is parked in TENSOR
// MEMORY (tcgen05.st / tcgen05.ld, 32 lanes x 32-bit columns per warp): it is a per-thread scratch that costs no
// registers and no shared-memory bandwidth while the second transform runs.
//
// Shared-memory planes are stored as 128-byte column tiles with the 16-byte chunk index XOR-ed with the row index
// (the layout a SWIZZLE_128B tensor-map copy produces): rows along a line of 8 lanes and columns along a line of 8
// lanes both hit eight different bank groups.
#pragma once
#include "common.cuh"
#include "state_kernels.cuh"
#include "plane_common.cuh"
#include "line_codelets.cuh"
#include <utility>
#include <type_traits>

// plane of N1 rows x N2 columns of 16-byte elements (columns = the contiguous global index)
template <int N1, int N2>
struct PlaneL {
    static constexpr int NT = (N2 + 7) / 8;                       // 128-byte column tiles
    static constexpr int TS = ((N1 * 8 + 63) / 64) * 64;          // elements per tile, 1024-byte aligned
    static constexpr int SIZE = NT * TS;
    __host__ __device__ static constexpr int idx(int row, int col) { return (col >> 3) * TS + row * 8 + ((col ^ row) & 7); }
};

// ---- explicit shared-memory addressing: 32-bit shared addresses, the constant part of every offset as an immediate ----
// byte address of point e of this thread's line in a plane that starts at `plane` (1024-byte aligned):
//     (B ^ ((e & 7) << 4)) + IMM(e),     B = plane + line part (below), one register per plane family;
//   ROWS (the line runs along the rows, at column `line`):   B = plane + tile(line) + ((line & 7) << 4),  IMM(e) = 128 e
//   !ROWS (the line runs along the columns, at row `line`):  B = plane + 128 line + ((line & 7) << 4),    IMM(e) = (e >> 3) TS 16
template <bool ROWS, int TS>
struct LineAddr {
    static __device__ __forceinline__ unsigned base(unsigned plane, int line)
    {
        return plane + (ROWS ? (unsigned)(line >> 3) * (TS * 16) : (unsigned)line * 128u) + ((unsigned)(line & 7) << 4);
    }
    __host__ __device__ static constexpr int k16(int e) { return (e & 7) << 4; }
    __host__ __device__ static constexpr int imm(int e) { return ROWS ? 128 * e : (e >> 3) * TS * 16; }
};
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
template <int K16, int IMM>
__device__ __forceinline__ double lds_f64(unsigned b)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(b ^ (unsigned)K16), "n"(IMM));
    return v;
}
template <int K16, int IMM>
__device__ __forceinline__ double2 lds_v2(unsigned b)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(v.x), "=d"(v.y) : "r"(b ^ (unsigned)K16), "n"(IMM));
    return v;
}
template <int K16, int IMM>
__device__ __forceinline__ void sts_f64(unsigned b, double v)
{
    asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(b ^ (unsigned)K16), "n"(IMM), "d"(v) : "memory");
}
// compile-time loop: f(std::integral_constant<int, I>) for I = 0 .. N-1
template <class F, int... I>
__device__ __forceinline__ void static_for_impl(F&& f, std::integer_sequence<int, I...>) { (f(std::integral_constant<int, I>{}), ...); }
template <int N, class F>
__device__ __forceinline__ void static_for(F&& f) { static_for_impl(f, std::make_integer_sequence<int, N>{}); }
// the points of a line in the order the pointwise loops visit them: e & 7 major, so that the XOR-ed address bases of
// a group of points (same e & 7) are formed once
__host__ __device__ constexpr int line_ord(int i, int n)
{
    int c = 0;
    for (int k = 0; k < 8; ++k)
        for (int e = k; e < n; e += 8) { if (c == i) return e; ++c; }
    return 0;
}

__device__ __forceinline__ double flip(double x, unsigned sgn) { return __hiloint2double(__double2hiint(x) ^ (int)sgn, __double2loint(x)); }

// ---- tensor memory as a per-thread scratch: warp w owns lanes 32 (w % 4) .. + 31, a thread one lane; a double is two
// 32-bit columns.  Allocation by warp 0 (power of two >= 32 columns), address published through shared memory. ----
template <int NCOLS>
__device__ __forceinline__ unsigned tmem_alloc(unsigned* s_slot, int warp)
{
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_slot)), "n"(NCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    return *(volatile unsigned*)s_slot;
}
template <int NCOLS>
__device__ __forceinline__ void tmem_free(unsigned taddr, int warp)
{
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(NCOLS) : "memory");
}
__device__ __forceinline__ void tmem_st4(unsigned taddr, double a, double b, double c, double d)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
                 "r"(__double2loint(a)), "r"(__double2hiint(a)), "r"(__double2loint(b)), "r"(__double2hiint(b)),
                 "r"(__double2loint(c)), "r"(__double2hiint(c)), "r"(__double2loint(d)), "r"(__double2hiint(d)) : "memory");
}
__device__ __forceinline__ void tmem_ld4(unsigned taddr, double& a, double& b, double& c, double& d)
{
    int r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr) : "memory");
    a = __hiloint2double(r[1], r[0]); b = __hiloint2double(r[3], r[2]);
    c = __hiloint2double(r[5], r[4]); d = __hiloint2double(r[7], r[6]);
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// N doubles of this thread (N % 4 == 0) back into registers, in the order they were parked
template <int N>
__device__ __forceinline__ void tmem_load_line(unsigned taddr, double (&v)[N])
{
#pragma unroll
    for (int c = 0; c < N / 4; ++c) tmem_ld4(taddr + 8 * c, v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
    tmem_wait_ld();
}
// columns of tensor memory a CTA of `warps` warps needs for one line of n doubles per thread (warps sharing a lane
// quadrant sit side by side), rounded up to a power of two >= 32
constexpr int tmem_cols(int warps, int n)
{
    const int need = ((warps + 3) / 4) * 2 * n;
    int c = 32;
    while (c < need) c *= 2;
    return c;
}

// ---- TMA (cp.async.bulk.tensor): one thread loads a whole [rows][128 bytes] plane tile, SWIZZLE_128B, completing on an mbarrier ----
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_tile(unsigned dst, const CUtensorMap* tm, unsigned long long* bar, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

struct LaneRole {
    int j, s, p;            // line within the task (0..7), spin component (0 up, 1 down), part (0 re, 1 im)
    unsigned pm, sm;        // sign-bit masks: sp = -1 for the imaginary part, ss = -1 for the down component (else +1)
    __device__ __forceinline__ void init()
    {
        const int lane = threadIdx.x & 31, c = lane >> 3;
        j = lane & 7; s = c >> 1; p = c & 1;
        pm = p ? 0x80000000u : 0u; sm = s ? 0x80000000u : 0u;
    }
};

// ------------------------------------------------------------------------------------------------
// T_axis phi of one 2-spinor on 8 lines, this lane's (spin, part) in "lane representation":
//     result at point line_ord(i) = (value parked at position i of the tensor-memory line `tr`) + cc[i].
//   bw  : address base (LineAddr::base) of the pair's UP component plane; the down plane follows SZB bytes later
//   bp  : address base of the axis' first potential plane P1 = (-M / 2 dx^2, A / dx); P2 = (w1 / dx, w2 / dx) follows
//         SZB bytes later (compact potentials of B_axis = A + (sigma x W)_axis / 2, see plane_common.cuh);
//         VLOC: V1 = (U + lap M / 2, S_x) and V2 = (S_y, S_z) follow at VOFF, VOFF + SZB: V_loc phi is included
//   cj  : 0x80000000 for the v pair (phi = conj v), else 0.  The planes hold the RAW components.  Conjugation is not
//         applied to the data: the imaginary-part lanes of the v pair carry -Im phi ("lane value = sigma x true value",
//         sigma = -1 for them), which every linear step preserves; in the pointwise products a coefficient that joins
//         an im lane with a re lane changes sign (cj is XOR-ed into its sign mask), and the caller maps the result
//         back: for the v pair -conj(h phi) = -(lane value) for both parts.
//   mid(): called once between the two codelets (barrier waits and prefetch issue sit behind the first transform)
// ------------------------------------------------------------------------------------------------
template <int N, int AXIS, bool ROWS, int TS, int SZB, bool VLOC, int VOFF, class Mid>
__device__ __forceinline__ void line_task6(unsigned bw, unsigned bp, unsigned cj, const LaneRole& ln, unsigned tr,
                                           double (&cc)[N], Mid mid)
{
    typedef LineAddr<ROWS, TS> LA;
    static_assert(N % 4 == 0, "lines are parked in tensor memory four points at a time");
    // this lane's part and the other part of its own component; same part / other part of the other spin component
    const unsigned bx = bw + (ln.s ? SZB : 0) + 8u * ln.p, bxo = bx ^ 8u;
    const unsigned bq = bw + (ln.s ? 0 : SZB) + 8u * ln.p, bqo = bq ^ 8u;
    double g[N], q[N];
    {
        double x[N], a[N], b[N];
        static_for<N>([&](auto ec) {
            constexpr int e = decltype(ec)::value;
            x[e] = lds_f64<LA::k16(e), LA::imm(e)>(bx);
        });
        LineCodelet<N>::inner(x, a, b);
        // sign mask of the coefficients of products with "other part" values (index 1, 3): sp and the conjugation
        const unsigned m13 = ln.pm ^ cj;
        // points in groups of 4 (in visiting order): all loads and shuffles of a group are issued before its arithmetic,
        // so that their latencies overlap; the group's four r1 values go to tensor memory with one store
        static_for<N / 4>([&](auto gc) {
            constexpr int g0 = 4 * decltype(gc)::value;
            double2 pa[4], pb[4], v1[4], v2[4];
            double f0[4], f1[4], f2[4], f3[4], a1[4], a2[4], a3[4], rr[4];
            static_for<4>([&](auto jc) {
                constexpr int jj = decltype(jc)::value, e = line_ord(g0 + jj, N);
                constexpr int K = LA::k16(e), I = LA::imm(e);
                pa[jj] = lds_v2<K, I>(bp); pb[jj] = lds_v2<K, I + SZB>(bp);
                f0[jj] = lds_f64<K, I>(bx); f1[jj] = lds_f64<K, I>(bxo);
                f2[jj] = f3[jj] = 0.0;
                if (AXIS != 1 || VLOC) f2[jj] = lds_f64<K, I>(bq);
                if (AXIS != 0 || VLOC) f3[jj] = lds_f64<K, I>(bqo);
                if (VLOC) { v1[jj] = lds_v2<K, I + VOFF>(bp); v2[jj] = lds_v2<K, I + VOFF + SZB>(bp); }
                a1[jj] = __shfl_xor_sync(0xffffffffu, a[e], 8);                       // other part, same spin
                a2[jj] = a3[jj] = 0.0;
                if (AXIS != 1) a2[jj] = __shfl_xor_sync(0xffffffffu, a[e], 16);       // same part, other spin
                if (AXIS != 0) a3[jj] = __shfl_xor_sync(0xffffffffu, a[e], 24);       // other part, other spin
            });
            static_for<4>([&](auto jc) {
                constexpr int jj = decltype(jc)::value, e = line_ord(g0 + jj, N);
                double r, gg;
                // (-i B t)_(s, p) with sp = +1 (re) / -1 (im), ss = +1 (up) / -1 (down); the signs are sign-bit flips
                if (AXIS == 0) {            // b_ss = A - ss w1, b01 = -i w2:   sp b_ss t1 - ss w2 t2
                    const double bs = flip(pa[jj].y - flip(pb[jj].x, ln.sm), m13), w = flip(pb[jj].y, ln.sm ^ 0x80000000u);
                    r = fma(bs, a1[jj], w * a2[jj]); gg = fma(bs, f1[jj], w * f2[jj]);
                } else if (AXIS == 1) {     // b_ss = A + ss w1, b01 = -w2:     sp (b_ss t1 - w2 t3)
                    const double bs = flip(pa[jj].y + flip(pb[jj].x, ln.sm), m13), w = flip(pb[jj].y, m13 ^ 0x80000000u);
                    r = fma(bs, a1[jj], w * a3[jj]); gg = fma(bs, f1[jj], w * f3[jj]);
                } else {                    // b_ss = A, b01 = w1 + i w2:       sp (A t1 + w1 t3) + ss w2 t2
                    const double bs = flip(pa[jj].y, m13), w1 = flip(pb[jj].x, m13), w2 = flip(pb[jj].y, ln.sm);
                    r = fma(bs, a1[jj], fma(w1, a3[jj], w2 * a2[jj])); gg = fma(bs, f1[jj], fma(w1, f3[jj], w2 * f2[jj]));
                }
                r = fma(pa[jj].x, b[e], r);
                if (VLOC) {                 // (U' + ss S_z) f0 + S_x f2 + ss sp S_y f3
                    r = fma(v1[jj].x + flip(v2[jj].y, ln.sm), f0[jj], r);
                    r = fma(v1[jj].y, f2[jj], r);
                    r = fma(flip(v2[jj].x, ln.sm ^ m13), f3[jj], r);
                }
                rr[jj] = r; g[e] = gg; q[e] = pa[jj].x * f0[jj];
            });
            tmem_st4(tr + 2 * g0, rr[0], rr[1], rr[2], rr[3]);
        });
        tmem_wait_st();
    }
    mid();
    double c[N];
    LineCodelet<N>::outer(g, q, c);
#pragma unroll
    for (int i = 0; i < N; ++i) cc[i] = c[line_ord(i, N)];
}

// staging of one axis' compact potentials into two swizzled double2 planes (scaled: D = D~ / dx, D2 = D~2 / dx^2)
__device__ __forceinline__ void put_pots(double2* P1, double2* P2, int si, double M, double A, double w1, double w2, double idx1, double idx2)
{
    P1[si] = make_double2(-0.5 * M * idx2, A * idx1);
    P2[si] = make_double2(0.5 * w1 * idx1, 0.5 * w2 * idx1);
}

// ------------------------------------------------------------------------------------------------
// H-apply, yz-planes:  W = [V_loc + T_y + T_z] X  (h of PAPER.md Eq. 12 without its x lines), with PAIRING also the
// pairing block of Eq. 11 (mu = 0): (H psi)_u += Delta (v_dn, -v_up), (H psi)_v += conj(Delta) (-u_dn, u_up).   grid (nx, G).
// A unit = NCOMP components (4: a state, 2: one 2-spinor) of one state on this CTA's plane.  Warps [0, NWY) run the y
// lines of the unit, warps [NWY, NWY + NWZ) its z lines at the same time; the z warps leave T_z phi + V_loc phi in
// the `oz` planes, the y warps add T_y phi, map the v pair back (-conj) and store W with row-contiguous 16-byte pairs.
// No CTA-wide barrier in the unit loop: mbarriers F[buf] ("unit landed": cp.async arrivals), E[buf] ("everyone is
// done with the unit in buf") and Z ("T_z of this unit is in the oz planes").
// shared: phi[2][NCOMP][SIZE] | oz[NCOMP][SIZE] | P1y P2y P1z P2z V1 V2 V3 [SIZE] (double2; V3 = Delta)
// ------------------------------------------------------------------------------------------------
template <int NY, int NZ, int NCOMP>
struct YZGeom {
    typedef PlaneL<NY, NZ> PL;
    static constexpr int NPAIR = NCOMP / 2, UPS = 4 / NCOMP;
    static constexpr int NTY = (NZ + 7) / 8, NTZ = (NY + 7) / 8;
    static constexpr int NWY = NPAIR * NTY, NWZ = NPAIR * NTZ, NW = NWY + NWZ;
    static constexpr size_t SMEM = 16 * (size_t)PL::SIZE * (2 * NCOMP + NCOMP + (NCOMP == 4 ? 7 : 6)) + 1024;   // V3 = Delta only with whole states; + alignment slack
    static constexpr int TCOLS = tmem_cols(NW, NY > NZ ? NY : NZ);
};

template <int NY, int NZ, int NCOMP, int MAXR, bool PAIRING>
__global__ void __maxnreg__(MAXR) k6_happly_yz(const __grid_constant__ HArgs a)
{
    static_assert(!PAIRING || NCOMP == 4, "the pairing block needs the whole state in the unit");
    typedef YZGeom<NY, NZ, NCOMP> G;
    typedef typename G::PL PL;
    constexpr int NPTS = NY * NZ, SZ = PL::SIZE, TS = PL::TS, SZB = SZ * 16;
    constexpr int NPAIR = G::NPAIR, UPS = G::UPS, NTHR = G::NW * 32, NMAX = NY > NZ ? NY : NZ;
    extern __shared__ unsigned char smem_raw[];
    const unsigned s_raw = smem_u32(smem_raw), s_phi = (s_raw + 1023u) & ~1023u;
    cplx* phi = (cplx*)(smem_raw + (s_phi - s_raw));
    cplx* oz = phi + 2 * NCOMP * SZ;
    double2* P1y = oz + NCOMP * SZ;
    double2 *P2y = P1y + SZ, *P1z = P2y + SZ, *P2z = P1z + SZ, *V1 = P2z + SZ, *V2 = V1 + SZ, *V3 = V2 + SZ;
    const unsigned s_oz = s_phi + 2 * NCOMP * SZB, s_py = s_oz + NCOMP * SZB, s_pz = s_py + 2 * SZB;
    __shared__ unsigned long long s_bar[5];
    __shared__ unsigned s_tmem;
    unsigned long long *barF = s_bar, *barE = s_bar + 2, *barZ = s_bar + 4;
    const int nxyz = a.L.nxyz, gbase = blockIdx.x * NPTS;
    const double* pot = a.pot;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // warp-uniform for the compiler: the role branch below does not diverge
    if (threadIdx.x == 0) {
        mbar_init(barF, 1); mbar_init(barF + 1, 1);               // "unit landed": one arrival (expect_tx) + the TMA's bytes
        mbar_init(barE, NTHR); mbar_init(barE + 1, NTHR);
        mbar_init(barZ, G::NWZ * 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const unsigned tbase = tmem_alloc<G::TCOLS>(&s_tmem, warp);     // includes a CTA-wide barrier
    const unsigned tr = tbase + ((unsigned)(warp & 3) << 21) + (unsigned)(warp >> 2) * (2 * NMAX);
    const int nunits = a.ns * UPS;
    // one thread stages a unit: NCOMP x NT tensor-map tile copies ([NY rows][128 bytes], hardware-swizzled)
    auto issue = [&](int u, int buf) {
        if (threadIdx.x != 0) return;
        mbar_expect_tx(barF + buf, NCOMP * PL::NT * NY * 128);
#pragma unroll
        for (int c = 0; c < NCOMP; ++c)
#pragma unroll
            for (int t = 0; t < PL::NT; ++t)
                tma_load_tile(s_phi + ((buf * NCOMP + c) * SZ + t * TS) * 16, &a.tmX, barF + buf, 16 * t, 0, (int)blockIdx.x, u * NCOMP + c);
    };
    int u = blockIdx.y;
    if (u < nunits) issue(u, 0);
    {
        const double i1 = 1.0 / a.L.dx, i2 = i1 * i1;
        for (int p = threadIdx.x; p < NPTS; p += NTHR) {
            const int y = p / NZ, z = p - y * NZ, si = PL::idx(y, z), gi = gbase + p;
            const double M = pot[(size_t)P_M * nxyz + gi];
            const double Wx = pot[(size_t)(P_W + 0) * nxyz + gi], Wy = pot[(size_t)(P_W + 1) * nxyz + gi], Wz = pot[(size_t)(P_W + 2) * nxyz + gi];
            put_pots(P1y, P2y, si, M, pot[(size_t)(P_A + 1) * nxyz + gi], Wx, Wz, i1, i2);
            put_pots(P1z, P2z, si, M, pot[(size_t)(P_A + 2) * nxyz + gi], Wy, Wx, i1, i2);
            double v[6]; load_vloc(pot, nxyz, gi, v);
            V1[si] = make_double2(v[0], v[1]); V2[si] = make_double2(v[2], v[3]);
            if (PAIRING) V3[si] = make_double2(v[4], v[5]);
        }
    }
    __syncthreads();

    const bool ywarp = warp < G::NWY;
    const int wl = ywarp ? warp : warp - G::NWY;
    const int pr = wl / (ywarp ? G::NTY : G::NTZ), strip = wl - pr * (ywarp ? G::NTY : G::NTZ);
    LaneRole ln; ln.init();
    const int nlines = ywarp ? NZ : NY;
    const int line_raw = 8 * strip + ln.j;
    const bool valid = line_raw < nlines;
    const int line = valid ? line_raw : nlines - 1;
    typedef LineAddr<true, TS> LAY;                                  // y lines: along the rows, at column z = line
    typedef LineAddr<false, TS> LAZ;                                 // z lines: along the columns of row y = line
    const unsigned b_pot = ywarp ? LAY::base(s_py, line) : LAZ::base(s_pz, line);
    const unsigned b_oz = (ywarp ? LAY::base(s_oz, line) : LAZ::base(s_oz, line)) + (2 * pr + ln.s) * SZB + 8u * ln.p;

    for (int it = 0; u < nunits; u += a.G, ++it) {
        const int buf = it & 1;
        mbar_wait(barF + buf, (it >> 1) & 1);                    // unit u has landed
        const int st = u / UPS, pg = u - st * UPS;
        const int pair = pg * NPAIR + pr;                        // 0: u pair, 1: v pair (phi = conj v)
        const unsigned cj = pair ? 0x80000000u : 0u;
        const unsigned s_unit = s_phi + buf * NCOMP * SZB;
        auto mid = [&]() {
            if (it >= 1) mbar_wait(barE + (buf ^ 1), ((it - 1) >> 1) & 1);    // unit u - G: oz and X[buf ^ 1] are free
            if (u + a.G < nunits) issue(u + a.G, buf ^ 1);
        };
        if (!ywarp) {
            // ---- z lines: T_z phi + V_loc phi -> oz ----
            double cc[NZ], r1[NZ];
            line_task6<NZ, 2, false, TS, SZB, true, 2 * SZB>(LAZ::base(s_unit + 2 * pr * SZB, line), b_pot, cj, ln, tr, cc, mid);
            tmem_load_line<NZ>(tr, r1);
            if (valid)
                static_for<NZ>([&](auto ic) {
                    constexpr int i = decltype(ic)::value, e = line_ord(i, NZ);
                    sts_f64<LAZ::k16(e), LAZ::imm(e)>(b_oz, r1[i] + cc[i]);
                });
            mbar_arrive(barZ);
        } else {
            // ---- y lines; finish W ----
            double cc[NY], r1[NY];
            line_task6<NY, 1, true, TS, SZB, false, 0>(LAY::base(s_unit + 2 * pr * SZB, line), b_pot, cj, ln, tr, cc, mid);
            tmem_load_line<NY>(tr, r1);
            mbar_wait(barZ, it & 1);
            double* Wg = (double*)(a.W + ((size_t)st * 4 + 2 * pair + ln.s) * nxyz + gbase + line) + ln.p;
            // pairing block (Eq. 11, mu = 0): u: + Delta (v_dn, -v_up), v: + conj(Delta) (-u_dn, u_up); partner =
            // component (other pair, other spin): u pair ss (Dr o2 - sp Di o3), v pair -ss (Dr o2 + sp Di o3)
            const unsigned b_o = LAY::base(s_unit + (2 * (1 - pair) + (1 - ln.s)) * SZB, line) + 8u * ln.p;
            const unsigned fa = pair ? (ln.sm ^ 0x80000000u) : ln.sm, fb = pair ? ln.pm : (ln.pm ^ 0x80000000u);
            static_for<NY>([&](auto ic) {
                constexpr int i = decltype(ic)::value, e = line_ord(i, NY);
                constexpr int K = LAY::k16(e), I = LAY::imm(e);
                // the v pair: -conj(h phi) = -(lane value) for both parts
                double t = flip(r1[i] + cc[i] + lds_f64<K, I>(b_oz), cj);
                if (PAIRING) {
                    const double2 dl = lds_v2<K, I + 6 * SZB>(b_pot);
                    const double o2 = lds_f64<K, I>(b_o), o3 = lds_f64<K, I>(b_o ^ 8u);
                    t += flip(fma(flip(dl.y, fb), o3, dl.x * o2), fa);
                }
                if (valid) __stcg(Wg + (size_t)e * NZ * 2, t);
            });
        }
        mbar_arrive(barE + buf);                                 // this thread is done with unit u
    }
    tmem_free<G::TCOLS>(tbase, warp);
}

// ------------------------------------------------------------------------------------------------
// H-apply, xz-planes:  W += T_x X (+ pairing block with PAIRING: PAPER.md Eq. 11, mu = 0:  (H psi)_u = h u + Delta (v_dn, -v_up),
// (H psi)_v = -conj(h conj v) + conj(Delta) (-u_dn, u_up));  eta_part[st * ny + iy] = dV Re <X|W> over the plane.
// grid (ny, G).  A unit = one state; every warp runs one strip of 8 x lines of one 2-spinor per unit; W is read from
// and written to global memory (row-contiguous 16-byte pairs) in the final loop, all loads in flight at once.
// mbarriers F[buf] / E[buf] per half as in k6_happly_yz.   shared: phi[NH][2][4][SIZE] | P1x P2x D [SIZE] | red[NH][2][NWH]
// ------------------------------------------------------------------------------------------------
// NH = units (states) a CTA works on at the same time: each "half" of NW / NH warps runs its own unit pipeline
// (own buffers and mbarriers) and shares the staged potentials; 2 where the planes are small enough (edges <= 24).
template <int NX, int NZ>
struct XZGeom {
    typedef PlaneL<NX, NZ> PL;
    static constexpr int NTX = (NZ + 7) / 8, NWH = 2 * NTX;
    static constexpr int NH = (NWH <= 6 && 16 * (size_t)PL::SIZE * (2 * 2 * 4 + 3) + 1024 <= 180 * 1024) ? 2 : 1;
    static constexpr int NW = NH * NWH;
    static constexpr size_t SMEM = 16 * (size_t)PL::SIZE * (NH * 2 * 4 + 3) + 1024;
    static constexpr int TCOLS = tmem_cols(NW, NX);
};

template <int NX, int NZ, int MAXR, bool PAIRING>
__global__ void __maxnreg__(MAXR) k6_happly_xz(const __grid_constant__ HArgs a)
{
    typedef XZGeom<NX, NZ> G;
    typedef typename G::PL PL;
    constexpr int NPTS = NX * NZ, SZ = PL::SIZE, TS = PL::TS, SZB = SZ * 16;
    constexpr int NW = G::NW, NTHR = NW * 32, NH = G::NH, NWH = G::NWH, NTHRH = NWH * 32;
    extern __shared__ unsigned char smem_raw[];
    const unsigned s_raw = smem_u32(smem_raw), s_phi = (s_raw + 1023u) & ~1023u;
    cplx* phi = (cplx*)(smem_raw + (s_phi - s_raw));
    double2* P1x = phi + NH * 2 * 4 * SZ;
    double2 *P2x = P1x + SZ, *Dl = P2x + SZ;
    const unsigned s_px = s_phi + NH * 2 * 4 * SZB;
    __shared__ double s_red[2 * NW];
    __shared__ unsigned long long s_bar[4 * NH];
    __shared__ unsigned s_tmem;
    const int nxyz = a.L.nxyz, gs = a.L.ny * NZ, gb = blockIdx.x * NZ;
    const double* pot = a.pot;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int half = warp / NWH, wh = warp - half * NWH;
    const bool leader = threadIdx.x == half * NTHRH;                  // first thread of the half: stages units, writes eta
    unsigned long long *barF = s_bar + 4 * half, *barE = barF + 2;
    double* red = s_red + 2 * NWH * half;
    if (threadIdx.x == 0) {
        for (int h = 0; h < NH; ++h) {
            mbar_init(s_bar + 4 * h, 1); mbar_init(s_bar + 4 * h + 1, 1);
            mbar_init(s_bar + 4 * h + 2, NTHRH); mbar_init(s_bar + 4 * h + 3, NTHRH);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const unsigned tbase = tmem_alloc<G::TCOLS>(&s_tmem, warp);
    const unsigned tr = tbase + ((unsigned)(warp & 3) << 21) + (unsigned)(warp >> 2) * (2 * NX);
    const int nunits = a.ns, ustep = a.G * NH;
    const unsigned s_half = s_phi + half * 2 * 4 * SZB;
    // one thread per half stages a unit: 4 x NT tensor-map tile copies ([NX rows at stride ny nz][128 bytes], hardware-swizzled)
    auto issue = [&](int u, int buf) {
        if (!leader) return;
        mbar_expect_tx(barF + buf, 4 * PL::NT * NX * 128);
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int t = 0; t < PL::NT; ++t)
                tma_load_tile(s_half + ((buf * 4 + c) * SZ + t * TS) * 16, &a.tmX, barF + buf, 16 * t, (int)blockIdx.x, 0, u * 4 + c);
    };
    auto flush_eta = [&](int uprev, int it_prev) {               // leader: fixed-order sum of the warps' partials
        double s = 0.0;
        for (int w = 0; w < NWH; ++w) s += red[(it_prev & 1) * NWH + w];
        a.eta_part[(size_t)uprev * a.L.ny + blockIdx.x] = s * a.L.dV;
    };
    int u = blockIdx.y * NH + half, uprev = -1;
    if (u < nunits) issue(u, 0);
    {
        const double i1 = 1.0 / a.L.dx, i2 = i1 * i1;
        for (int p = threadIdx.x; p < NPTS; p += NTHR) {
            const int x = p / NZ, z = p - x * NZ, si = PL::idx(x, z), gi = gb + x * gs + z;
            put_pots(P1x, P2x, si, pot[(size_t)P_M * nxyz + gi], pot[(size_t)(P_A + 0) * nxyz + gi],
                     pot[(size_t)(P_W + 1) * nxyz + gi], pot[(size_t)(P_W + 2) * nxyz + gi], i1, i2);
            Dl[si] = make_double2(pot[(size_t)P_DELTA * nxyz + gi], pot[(size_t)(P_DELTA + 1) * nxyz + gi]);
        }
    }
    __syncthreads();

    const int pr = wh / G::NTX, strip = wh - pr * G::NTX;        // pr = pair: 0 the u pair, 1 the v pair (phi = conj v)
    LaneRole ln; ln.init();
    const int line_raw = 8 * strip + ln.j;
    const bool valid = line_raw < NZ;
    const int line = valid ? line_raw : NZ - 1;
    typedef LineAddr<true, TS> LA;                                   // x lines: along the rows, at column z = line
    const unsigned b_pot = LA::base(s_px, line);
    const unsigned cj = pr ? 0x80000000u : 0u;
    // pairing partner: component (other pair, other spin);  u pair: ss (Dr o2 - sp Di o3),  v pair: -ss (Dr o2 + sp Di o3)
    const int oc = 2 * (1 - pr) + (1 - ln.s);
    const unsigned fa = pr ? (ln.sm ^ 0x80000000u) : ln.sm, fb = pr ? ln.pm : (ln.pm ^ 0x80000000u);
    int it = 0;
    for (; u < nunits; u += ustep, ++it) {
        const int buf = it & 1;
        mbar_wait(barF + buf, (it >> 1) & 1);
        const unsigned s_unit = s_half + buf * 4 * SZB;
        const unsigned b_w = LA::base(s_unit + 2 * pr * SZB, line);
        auto mid = [&]() {
            if (it >= 1) {
                mbar_wait(barE + (buf ^ 1), ((it - 1) >> 1) & 1);    // this half is done with unit u - ustep
                if (leader) flush_eta(uprev, it - 1);
            }
            if (u + ustep < nunits) {
                issue(u + ustep, buf ^ 1);
                // the next unit's W values of this thread's points: into L2 now, so that the loads below do not wait for
                // HBM while the ABM update streams beside this CTA
                const double* wn = (const double*)(a.W + ((size_t)(u + ustep) * 4 + 2 * pr + ln.s) * nxyz + gb + line) + ln.p;
#pragma unroll
                for (int i = 0; i < NX; ++i) asm volatile("prefetch.global.L2 [%0];" ::"l"(wn + (size_t)i * gs * 2));
            }
        };
        double cc[NX];
        line_task6<NX, 0, true, TS, SZB, false, 0>(b_w, b_pot, cj, ln, tr, cc, mid);
        double* Wg = (double*)(a.W + ((size_t)u * 4 + 2 * pr + ln.s) * nxyz + gb + line) + ln.p;
        double win[NX];                                              // all loads of W in flight before the first use
#pragma unroll
        for (int i = 0; i < NX; ++i) win[i] = __ldcg(Wg + (size_t)line_ord(i, NX) * gs * 2);
#pragma unroll
        for (int c = 0; c < NX / 4; ++c) {                           // cc <- the whole T_x phi part, mapped back for the v pair:
            double t0, t1, t2, t3;                                   // -conj(h phi) = -(lane value) for both parts
            tmem_ld4(tr + 8 * c, t0, t1, t2, t3);
            tmem_wait_ld();
            cc[4 * c] = flip(t0 + cc[4 * c], cj); cc[4 * c + 1] = flip(t1 + cc[4 * c + 1], cj);
            cc[4 * c + 2] = flip(t2 + cc[4 * c + 2], cj); cc[4 * c + 3] = flip(t3 + cc[4 * c + 3], cj);
        }
        const unsigned b_x = b_w + (ln.s ? SZB : 0) + 8u * ln.p;     // this lane's raw component part
        const unsigned b_o = LA::base(s_unit + oc * SZB, line) + 8u * ln.p;
        double eta = 0.0;
        static_for<NX>([&](auto ic) {
            constexpr int i = decltype(ic)::value, e = line_ord(i, NX);
            constexpr int K = LA::k16(e), I = LA::imm(e);
            double w = win[i] + cc[i];
            if (PAIRING) {
                const double2 dl = lds_v2<K, I + 2 * SZB>(b_pot);
                const double o2 = lds_f64<K, I>(b_o), o3 = lds_f64<K, I>(b_o ^ 8u);
                w += flip(fma(flip(dl.y, fb), o3, dl.x * o2), fa);
            }
            if (valid) { __stcg(Wg + (size_t)e * gs * 2, w); eta = fma(lds_f64<K, I>(b_x), w, eta); }
        });
        for (int o = 16; o > 0; o >>= 1) eta += __shfl_xor_sync(0xffffffffu, eta, o);
        if ((threadIdx.x & 31) == 0) red[(it & 1) * NWH + wh] = eta;
        mbar_arrive(barE + buf);
        uprev = u;
    }
    __syncthreads();
    if (leader && uprev >= 0) flush_eta(uprev, it - 1);
    tmem_free<G::TCOLS>(tbase, warp);
}

// every register of the SM for a CTA of `warps` warps that runs without a neighbour: the register file is per
// sub-partition (16384 each), which ceil(warps / 4) warps share
__host__ __device__ constexpr int fft_full_regs(int warps)
{
    const int r = (16384 / (((warps + 3) / 4) * 32)) & ~7;
    return r > 255 ? 255 : r;
}
// The whole-state yz kernels (edges <= 24) live in their own translation unit, happly_yz_whole.cu, which build.py compiles
// with ptxas --register-usage-level=3: at 24^3 that schedule spills 84 instead of 260 bytes and runs 18.7 instead of 20.4 ms
// per step; every other kernel is faster at the default level (measured).
typedef void (*K6Kern)(HArgs);
template <int NY, int NZ> K6Kern k6_yz_whole();
