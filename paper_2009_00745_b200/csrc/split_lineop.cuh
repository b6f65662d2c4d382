// split_lineop.cuh -- the lattice line operator D_i, D2_i (Eqs. 48-50) as a BLOCK-DIAGONALISED circulant
// on the fp64 tensor cores ("v5" line operator).
//
// A line of N = R*H points, n = r + H*m (r < H, m < R).  The circulant y[n] = sum_n' c[n - n'] x[n'] is a
// circulant of size R in the coarse index m for every (r, r'); the REAL discrete Fourier transform of size R over
// m (cos / sin rows, thread-local: a thread holds the R points n = r + H*m of its row r) block-diagonalises it:
//     b_j[r'] = sum_m cos(2 pi j m / R) x[r' + H m],   e_j[r'] = sum_m sin(2 pi j m / R) x[r' + H m]
//     S_j = P_j b_j - Q_j e_j,   T_j = P_j e_j + Q_j b_j          (H x H real Toeplitz blocks P_j, Q_j)
//     y[r + H m] = sum_j cos(2 pi j m / R) S_j[r] + sin(2 pi j m / R) T_j[r]
//     P_j[d] = (w_j / R) sum_p cos(2 pi j p / R) c[d + H p],  Q_j likewise with sin;  w_j = 1 (j = 0, R/2) else 2.
// Only the H x H blocks go through DMMA: for H = 8 that is 2 (real j) or 8 (conjugate pair) m8n8k4 tiles per
// 8 data columns instead of (N/8)(N/4) for the full circulant -- 10 instead of 18 at N = 24, 12 instead of 32 at
// N = 32.  H = N (R = 1) is the plain circulant, used when N is not a multiple of 8.
// The transform is an exact algebraic identity (the paper's operator is unchanged; rounding order differs).
//
// "Spectral order" q = 0..R-1 of the R real values replacing the R points:  q = 0: b_0;  q = 2j-1, 2j: b_j, e_j
// (1 <= j < R/2);  q = R-1: b_{R/2} when R is even.
#pragma once
#include "common.cuh"

#define LISE_RMAX 8
// generic real-DFT coefficients: c_rdft[R][q][m]; filled by the host (lise.cu: upload_rdft)
__constant__ double c_rdft[LISE_RMAX + 1][LISE_RMAX][LISE_RMAX];

template <int N_>
struct LOp {
    static constexpr int N = N_;
    static constexpr int H = (N % 8 == 0 && N >= 16 && N / 8 <= LISE_RMAX) ? 8 : N;
    static constexpr int R = N / H, J = R / 2 + 1;
    static constexpr int NTH = (H + 7) / 8;          // row tiles of a block
    static constexpr int NKH = H / 4;                // k steps of a block
    static constexpr int NFR = 2 * NTH + NKH - 2;    // distinct Toeplitz fragments per (op, j, P|Q)
    static constexpr int ND = H + 8 * NTH - 1;       // table entries d = -(H-1) .. 8 NTH - 1
    static constexpr int TABSZ = 2 * J * 2 * ND;     // doubles: [op][j][P|Q][d]
    static constexpr int NPAIR = (R - 1) / 2;        // conjugate pairs j = 1..NPAIR
    static_assert(N % 4 == 0, "line length must be a multiple of 4");
};

__device__ __forceinline__ void dmma5(double (&d)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

// ---- thread-local real DFT over the R coarse points: fwd (points -> spectral order), inv (its transpose) ----
template <int R>
struct RDFT {
    static __device__ __forceinline__ void fwd(const double (&x)[R], double (&v)[R])
    {
#pragma unroll
        for (int q = 0; q < R; ++q) {
            double s = 0.0;
#pragma unroll
            for (int m = 0; m < R; ++m) s = fma(c_rdft[R][q][m], x[m], s);
            v[q] = s;
        }
    }
    static __device__ __forceinline__ void inv(const double (&a)[R], double (&y)[R])
    {
#pragma unroll
        for (int m = 0; m < R; ++m) {
            double s = 0.0;
#pragma unroll
            for (int q = 0; q < R; ++q) s = fma(c_rdft[R][q][m], a[q], s);
            y[m] = s;
        }
    }
};
template <>
struct RDFT<1> {
    static __device__ __forceinline__ void fwd(const double (&x)[1], double (&v)[1]) { v[0] = x[0]; }
    static __device__ __forceinline__ void inv(const double (&a)[1], double (&y)[1]) { y[0] = a[0]; }
};
template <>
struct RDFT<2> {
    static __device__ __forceinline__ void fwd(const double (&x)[2], double (&v)[2]) { v[0] = x[0] + x[1]; v[1] = x[0] - x[1]; }
    static __device__ __forceinline__ void inv(const double (&a)[2], double (&y)[2]) { y[0] = a[0] + a[1]; y[1] = a[0] - a[1]; }
};
#define LISE_SIN60 0.86602540378443864676
template <>
struct RDFT<3> {
    static __device__ __forceinline__ void fwd(const double (&x)[3], double (&v)[3])
    {
        const double s = x[1] + x[2];
        v[0] = x[0] + s; v[1] = fma(-0.5, s, x[0]); v[2] = LISE_SIN60 * (x[1] - x[2]);
    }
    static __device__ __forceinline__ void inv(const double (&a)[3], double (&y)[3])
    {
        const double u = fma(-0.5, a[1], a[0]), w = LISE_SIN60 * a[2];
        y[0] = a[0] + a[1]; y[1] = u + w; y[2] = u - w;
    }
};
template <>
struct RDFT<4> {
    static __device__ __forceinline__ void fwd(const double (&x)[4], double (&v)[4])
    {
        const double s02 = x[0] + x[2], s13 = x[1] + x[3];
        v[0] = s02 + s13; v[1] = x[0] - x[2]; v[2] = x[1] - x[3]; v[3] = s02 - s13;
    }
    static __device__ __forceinline__ void inv(const double (&a)[4], double (&y)[4])
    {
        const double p = a[0] + a[3], m = a[0] - a[3];
        y[0] = p + a[1]; y[1] = m + a[2]; y[2] = p - a[1]; y[3] = m - a[2];
    }
};

#define LISE_COS72 0.30901699437494742410
#define LISE_COS144 (-0.80901699437494742410)
#define LISE_SIN72 0.95105651629515357212
#define LISE_SIN144 0.58778525229247312917
template <>
struct RDFT<5> {                                   // spectral order b0, b1, e1, b2, e2
    static __device__ __forceinline__ void fwd(const double (&x)[5], double (&v)[5])
    {
        const double p14 = x[1] + x[4], m14 = x[1] - x[4], p23 = x[2] + x[3], m23 = x[2] - x[3];
        v[0] = x[0] + p14 + p23;
        v[1] = fma(LISE_COS72, p14, fma(LISE_COS144, p23, x[0]));
        v[2] = fma(LISE_SIN72, m14, LISE_SIN144 * m23);
        v[3] = fma(LISE_COS144, p14, fma(LISE_COS72, p23, x[0]));
        v[4] = fma(LISE_SIN144, m14, -LISE_SIN72 * m23);
    }
    static __device__ __forceinline__ void inv(const double (&a)[5], double (&y)[5])
    {
        const double A1 = fma(LISE_COS72, a[1], fma(LISE_COS144, a[3], a[0])), B1 = fma(LISE_SIN72, a[2], LISE_SIN144 * a[4]);
        const double A2 = fma(LISE_COS144, a[1], fma(LISE_COS72, a[3], a[0])), B2 = fma(LISE_SIN144, a[2], -LISE_SIN72 * a[4]);
        y[0] = a[0] + a[1] + a[3]; y[1] = A1 + B1; y[2] = A2 + B2; y[3] = A2 - B2; y[4] = A1 - B1;
    }
};
template <>
struct RDFT<6> {                                   // spectral order b0, b1, e1, b2, e2, b3
    static __device__ __forceinline__ void fwd(const double (&x)[6], double (&v)[6])
    {
        const double s03 = x[0] + x[3], d03 = x[0] - x[3], s14 = x[1] + x[4], d14 = x[1] - x[4], s25 = x[2] + x[5], d25 = x[2] - x[5];
        v[0] = s03 + s14 + s25; v[1] = fma(0.5, d14 - d25, d03); v[2] = LISE_SIN60 * (d14 + d25);
        v[3] = fma(-0.5, s14 + s25, s03); v[4] = LISE_SIN60 * (s14 - s25); v[5] = d03 - d14 + d25;
    }
    static __device__ __forceinline__ void inv(const double (&a)[6], double (&y)[6])
    {
        const double P = fma(-0.5, a[3], a[0]), Q = fma(0.5, a[1], -a[5]);
        const double sp = LISE_SIN60 * (a[2] + a[4]), sm = LISE_SIN60 * (a[2] - a[4]);
        y[0] = a[0] + a[1] + a[3] + a[5]; y[3] = a[0] - a[1] + a[3] - a[5];
        y[1] = P + Q + sp; y[2] = P - Q + sm; y[4] = P - Q - sm; y[5] = P + Q - sp;
    }
};
#define LISE_SQRT_HALF 0.70710678118654752440
template <>
struct RDFT<8> {                                   // spectral order b0, b1, e1, b2, e2, b3, e3, b4
    static __device__ __forceinline__ void fwd(const double (&x)[8], double (&v)[8])
    {
        const double s04 = x[0] + x[4], d04 = x[0] - x[4], s26 = x[2] + x[6], d26 = x[2] - x[6];
        const double s15 = x[1] + x[5], d15 = x[1] - x[5], s37 = x[3] + x[7], d37 = x[3] - x[7];
        const double se = s04 + s26, so = s15 + s37;
        const double u = LISE_SQRT_HALF * (d15 - d37), w = LISE_SQRT_HALF * (d15 + d37);
        v[0] = se + so; v[1] = d04 + u; v[2] = d26 + w; v[3] = s04 - s26;
        v[4] = s15 - s37; v[5] = d04 - u; v[6] = w - d26; v[7] = se - so;
    }
    static __device__ __forceinline__ void inv(const double (&a)[8], double (&y)[8])
    {
        const double p0 = a[0] + a[7], p1 = a[0] - a[7];
        const double e0 = p0 + a[3], e2 = p0 - a[3], o1 = p1 + a[4], o3 = p1 - a[4];
        const double s13 = a[1] + a[5], d13 = a[1] - a[5], s26 = a[2] + a[6], d26 = a[2] - a[6];
        const double t1 = LISE_SQRT_HALF * (d13 + s26), t3 = LISE_SQRT_HALF * (s26 - d13);
        y[0] = e0 + s13; y[4] = e0 - s13; y[2] = e2 + d26; y[6] = e2 - d26;
        y[1] = o1 + t1; y[5] = o1 - t1; y[3] = o3 + t3; y[7] = o3 - t3;
    }
};

// ---- Toeplitz fragments of one operator (op = 0: D, 1: D2) for this thread (g = lane / 4, t = lane % 4) ----
// fragment f <-> (2 r - kk) = f - (NKH - 1):  A[g][t] = P_j[(8 r + g) - (4 kk + t)]
template <int N>
struct Frags {
    typedef LOp<N> L;
    double P[L::J][L::NFR], Q[L::J][L::NFR];
    __device__ __forceinline__ void load(const double* __restrict__ tab, int op, int g, int t)
    {
#pragma unroll
        for (int j = 0; j < L::J; ++j)
#pragma unroll
            for (int f = 0; f < L::NFR; ++f) {
                const int d = 4 * (f - (L::NKH - 1)) + g - t;
                P[j][f] = tab[((op * L::J + j) * 2 + 0) * L::ND + d + L::H - 1];
                Q[j][f] = tab[((op * L::J + j) * 2 + 1) * L::ND + d + L::H - 1];
            }
    }
};

// acc[q][r] += block_j(op) v   for k step kk (compile-time after unrolling); v in spectral order
template <int N>
__device__ __forceinline__ void mma_blocks(double (&acc)[LOp<N>::R][LOp<N>::NTH][2], const Frags<N>& F,
                                           const double (&v)[LOp<N>::R], int kk)
{
    typedef LOp<N> L;
#pragma unroll
    for (int r = 0; r < L::NTH; ++r) {
        const int f = 2 * r - kk + L::NKH - 1;
        dmma5(acc[0][r], F.P[0][f], v[0]);
#pragma unroll
        for (int j = 1; j <= L::NPAIR; ++j) {
            const int qc = 2 * j - 1, qs = 2 * j;
            dmma5(acc[qc][r], F.P[j][f], v[qc]); dmma5(acc[qc][r], F.Q[j][f], -v[qs]);
            dmma5(acc[qs][r], F.P[j][f], v[qs]); dmma5(acc[qs][r], F.Q[j][f], v[qc]);
        }
        if (L::R % 2 == 0) dmma5(acc[L::R - 1][r], F.P[L::R / 2][f], v[L::R - 1]);
    }
}

template <int N>
__device__ __forceinline__ void zero_acc(double (&acc)[LOp<N>::R][LOp<N>::NTH][2])
{
#pragma unroll
    for (int q = 0; q < LOp<N>::R; ++q)
#pragma unroll
        for (int r = 0; r < LOp<N>::NTH; ++r) acc[q][r][0] = acc[q][r][1] = 0.0;
}

// spectral accumulators -> point values, in place: acc[m][r][c] = value at row H m + 8 r + g
template <int N>
__device__ __forceinline__ void post_transform(double (&acc)[LOp<N>::R][LOp<N>::NTH][2])
{
    typedef LOp<N> L;
#pragma unroll
    for (int r = 0; r < L::NTH; ++r)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            double a[L::R], y[L::R];
#pragma unroll
            for (int q = 0; q < L::R; ++q) a[q] = acc[q][r][c];
            RDFT<L::R>::inv(a, y);
#pragma unroll
            for (int m = 0; m < L::R; ++m) acc[m][r][c] = y[m];
        }
}
