// plane_common.cuh -- helpers shared by the plane-owner kernels (plane5_kernels.cuh).
//   * shared-memory planes are stored [n1][LD] with LD = n2 padded so that LD % 8 == 4 (in 16-byte units):
//     the operand addresses of a DMMA fragment load then fall into two conflict-free wavefronts;
//   * the potentials of a plane are staged once per launch in compact form (M, A_i, W/2);
//   * cp.async helpers for prefetching the next unit's wavefunction plane.
#pragma once
#include "common.cuh"
#include "state_kernels.cuh"

// Register budget of a plane-owner CTA that is to share its SM with the ABM update CTA (k5_update: 4 warps, one per
// SM sub-partition, <= LISE_UPD_REGS registers).  The register file is per sub-partition (16384 registers each), so
// the budget is per sub-partition too: (warps / 4) x 32 x R + 32 x LISE_UPD_REGS <= 16384.
#define LISE_UPD_REGS 80
__host__ __device__ constexpr int coresident_regs(int warps)
{
    const int r = ((16384 - 32 * LISE_UPD_REGS) / (((warps + 3) / 4) * 32)) & ~7;
    return r > 255 ? 255 : r;
}
__host__ __device__ constexpr int ldpad(int n) { return n + ((4 - n % 8) + 8) % 8; }

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NPENDING) : "memory"); }

// ---- shared-memory mbarriers: split arrive / wait, so that a warp signals "done" and runs on instead of stopping at a
// CTA-wide barrier (the plane kernels let their warps drift apart by up to one task) ----
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(s) : "memory");
}
// the executing thread's earlier cp.async copies arrive on the barrier when they have landed (count not incremented:
// the barrier's expected count includes this arrival)
__device__ __forceinline__ void mbar_arrive_cp_async(unsigned long long* bar)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(s) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 ::"r"(s), "r"(parity) : "memory");
}

// compact potentials of one plane for one axis, in shared memory (doubles, same padded layout as the planes)
//   B_i = A_i + (sigma x W)_i / 2:  x: b00 = A - hWy, b11 = A + hWy, b01 = (0, -hWz)
//                                   y: b00 = A + hWx, b11 = A - hWx, b01 = (-hWz, 0)
//                                   z: b00 = b11 = A,               b01 = (hWy, hWx)        (hW = W / 2)
struct AxisPot4 {
    const double* M;      // -(hbar^2 / 2m*) / 2
    const double* A;      // A_axis
    const double* w1;     // x: hWy   y: hWx   z: hWy
    const double* w2;     // x: hWz   y: hWz   z: hWx
};

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

// rows of the V_loc / pairing staging area pV (VSTAGE) and their source rows in the potential array
__device__ __forceinline__ void load_vloc(const double* __restrict__ pot, int nxyz, int gi, double (&v)[6])
{
    v[0] = pot[(size_t)P_ULOC * nxyz + gi];
    v[1] = pot[(size_t)(P_S + 0) * nxyz + gi]; v[2] = pot[(size_t)(P_S + 1) * nxyz + gi]; v[3] = pot[(size_t)(P_S + 2) * nxyz + gi];
    v[4] = pot[(size_t)P_DELTA * nxyz + gi];   v[5] = pot[(size_t)(P_DELTA + 1) * nxyz + gi];
}

