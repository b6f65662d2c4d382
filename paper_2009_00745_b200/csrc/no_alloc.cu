// no_alloc.cu -- lise_renormalize_static: the renormalisation of PAPER.md:L637 for callers that must not allocate.
//
// Who this is for.  A TDSLDA run is sized so that the wavefunctions and their multistep history fill the GPU
// (7 state arrays per species), and the application that owns those arrays usually took the memory through
// a pool of its own (torch's caching allocator, an MPI code's arena).  Such a caller has no spare bytes for a library to
// cudaMalloc, and a cudaMalloc / cudaFree pair in the middle of a time loop also stalls every stream of the device while
// the driver maps and unmaps memory.  Everything else in liblise.so goes through lise_create, which allocates; this one
// entry point does not: no context, no cudaMalloc / cudaFree, no allocating library routine.  The only memory it
// touches besides the caller's array is the fixed array below, which is part of the library image.
//
// Price of that: the array (LISE_STATIC_MAX_STATES doubles = 128 KB) sits on EVERY GPU that loads liblise.so, from the
// moment the CUDA module is loaded until the process exits, whether or not this call is ever made; a call is limited to
// LISE_STATIC_MAX_STATES states (larger sets: several calls on slices of the array); and all calls on one device share
// the array (see "sharing" below).
//
// The arithmetic is that of k_state_norms / k_state_scale (grid_kernels.cuh), which lise_params.renormalize uses on
// the context's own per-state scratch; the kernels are repeated here so that the existing path is not touched.
#include "common.cuh"
#include <mutex>

#if LISE_STATIC_MAX_STATES != 16384
#error "include/lise.h and no_alloc.cu disagree about LISE_STATIC_MAX_STATES"
#endif

// Scratch: norm[k] = dV sum |psi_k|^2 of the call in flight.  In HOST code the name g_static_norms is only a handle for
// the symbol (not a device address); host code gets the real address once per device from cudaGetSymbolAddress below.
static __device__ __align__(256) double g_static_norms[LISE_STATIC_MAX_STATES];

// one block per state; same summation order as k_state_norms, so the two paths agree bit for bit
__global__ void k_static_state_norms(const cplx* __restrict__ psi, size_t slen, double dV, double* __restrict__ nrm)
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
        nrm[blockIdx.x] = t * dV;          // plain store: the slot is overwritten, never accumulated into
    }
}
// psi_k <- psi_k / sqrt(norm[k]); a state that is identically zero (norm 0) is left as it is
__global__ void k_static_state_scale(cplx* __restrict__ psi, size_t slen, const double* __restrict__ nrm)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= slen) return;
    const double n = nrm[blockIdx.y];
    if (!(n > 0.0)) return;
    const double f = rsqrt(n);
    cplx* p = psi + (size_t)blockIdx.y * slen + i;
    const cplx v = *p;
    *p = cmk(v.x * f, v.y * f);
}

// ---- per-device set-up ---------------------------------------------------------------------------------------------
static const int kMaxDevices = 64;
static std::mutex g_setup_mutex;
static double* g_norms_addr[kMaxDevices];       // device address of g_static_norms on device d; null until set up there
static thread_local char t_err[256] = "";

// Device address of the scratch on the CURRENT device.  The first call on a device asks the runtime for it
// (cudaGetSymbolAddress loads this library's CUDA module on that device if it is not loaded yet); later calls read the
// cached pointer.  Each device has its own copy of the array at its own address, hence one slot per device.
static int static_scratch(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        snprintf(t_err, sizeof(t_err), "cudaGetDevice: %s", cudaGetErrorString(e));
        return LISE_ECUDA;
    }
    if (dev < 0 || dev >= kMaxDevices) {
        snprintf(t_err, sizeof(t_err), "device ordinal %d is outside the %d devices this entry point keeps a scratch address for", dev, kMaxDevices);
        return LISE_EUNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_norms_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_norms);
        if (e != cudaSuccess || !p) {
            snprintf(t_err, sizeof(t_err), "cudaGetSymbolAddress(g_static_norms) on device %d: %s", dev, cudaGetErrorString(e));
            return LISE_ECUDA;
        }
        g_norms_addr[dev] = (double*)p;
    }
    *out = g_norms_addr[dev];
    return LISE_OK;
}

extern "C" int lise_renormalize_static(void* psi_dev, int nstates, long long state_len, double dV, void* cuda_stream)
{
    t_err[0] = 0;
    if (nstates < 0 || state_len <= 0 || !(dV > 0.0) || !(dV < INFINITY) || (nstates > 0 && !psi_dev)) {
        snprintf(t_err, sizeof(t_err), "bad argument: psi_dev %p, nstates %d, state_len %lld, dV %g", psi_dev, nstates, state_len, dV);
        return LISE_EINVAL;
    }
    if (nstates > LISE_STATIC_MAX_STATES) {
        snprintf(t_err, sizeof(t_err), "nstates = %d is more than LISE_STATIC_MAX_STATES = %d, the size of the library's fixed scratch: "
                 "call once per slice of at most %d states", nstates, LISE_STATIC_MAX_STATES, LISE_STATIC_MAX_STATES);
        return LISE_EINVAL;
    }
    const size_t slen = (size_t)state_len;
    const size_t nbx = (slen + 255) / 256;
    if (nbx > 2147483647ull) {
        snprintf(t_err, sizeof(t_err), "state_len %lld is too long for one launch", state_len);
        return LISE_EINVAL;
    }
    if (nstates == 0) return LISE_OK;
    double* nrm = nullptr;
    const int rc = static_scratch(&nrm);
    if (rc != LISE_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cplx* psi = (cplx*)psi_dev;
    k_static_state_norms<<<nstates, 256, 0, st>>>(psi, slen, dV, nrm);
    k_static_state_scale<<<dim3((unsigned)nbx, nstates), 256, 0, st>>>(psi, slen, nrm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(t_err, sizeof(t_err), "kernel launch: %s", cudaGetErrorString(e));
        return LISE_ECUDA;
    }
    return LISE_OK;
}

extern "C" const char* lise_static_last_error(void) { return t_err; }
