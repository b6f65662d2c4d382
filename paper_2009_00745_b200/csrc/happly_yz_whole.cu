// happly_yz_whole.cu -- the FFT yz H-apply kernels that see whole states (every lattice of LISE_FFT_SHAPES in lise.cu with
// edges <= 24), in a translation unit of their own: build.py compiles this file with ptxas --register-usage-level=3
// (see fft_plane_kernels.cuh).  (ny, nz) pairs of the lattices (nx, ny, nz) lise.cu instantiates.
#include "fft_plane_kernels.cuh"

#define LISE_YZ_WHOLE(NY, NZ) \
    template <> K6Kern k6_yz_whole<NY, NZ>() { return k6_happly_yz<NY, NZ, 4, fft_full_regs(YZGeom<NY, NZ, 4>::NW), true>; }
LISE_YZ_WHOLE(8, 8) LISE_YZ_WHOLE(12, 12) LISE_YZ_WHOLE(16, 16) LISE_YZ_WHOLE(20, 20) LISE_YZ_WHOLE(24, 24)
LISE_YZ_WHOLE(8, 16) LISE_YZ_WHOLE(12, 8) LISE_YZ_WHOLE(12, 16)
