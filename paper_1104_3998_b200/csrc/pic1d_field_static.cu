// pic1d_field_static.cu -- pic1d_field_solve_static (include/pic1d_static.h): the global-memory Poisson + E
// kernel of the step (k_field in pic1d_grid.cuh; Eq. 1-2) for callers that cannot
// create device memory.  k_field keeps its two running sums S and T in the caller's workspace; this variant keeps
// them in a fixed array compiled into the library, so the call needs no cudaMalloc, no workspace and no handle.
// Self-contained on purpose: it shares no code with the step's path and changes nothing there.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/pic1d.h"
#include "../../include/pic1d_static.h"

// The scratch: S in [0, MAX), T in [MAX, 2 MAX).  One copy per device that has this module loaded, alive until
// the process exits.  In HOST code the name below is only a handle for cudaGetSymbolAddress -- it is not a
// device address and must never be handed to a kernel as one.
static __device__ __align__(256) double g_field_scratch[2 * PIC1D_FIELD_STATIC_MAX_CELLS];

namespace {

__device__ __forceinline__ double fs_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// sum over the block, returned to every thread (blockDim.x a multiple of 32, at most 1024)
__device__ double fs_block_sum(double v) {
    __shared__ double s_r[32];
    __shared__ double s_out;
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    v = fs_warp_sum(v);
    if (lane == 0) s_r[wp] = v;
    __syncthreads();
    if (wp == 0) {
        double t = lane < (int)(blockDim.x >> 5) ? s_r[lane] : 0.0;
        t = fs_warp_sum(t);
        if (lane == 0) s_out = t;
    }
    __syncthreads();
    const double r = s_out;
    __syncthreads();
    return r;
}

// dst[i] = sum_{m <= i} src(m), i < n: every thread sums a contiguous chunk, the chunk totals are scanned with
// shuffles, then every thread walks its chunk again.  Ends with a barrier, so dst is visible to the whole block.
template <class F>
__device__ void fs_block_scan(F src, double* dst, int n) {
    __shared__ double s_w[32];
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5, nw = blockDim.x >> 5;
    const int ch = (n + blockDim.x - 1) / blockDim.x;
    const int b = tid * ch, e = min(b + ch, n);
    double tot = 0.0;
    for (int i = b; i < e; ++i) tot += src(i);
    double inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[wp] = inc;
    __syncthreads();
    if (wp == 0) {
        const double t = lane < nw ? s_w[lane] : 0.0;
        double ti = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double u = __shfl_up_sync(0xffffffffu, ti, o);
            if (lane >= o) ti += u;
        }
        s_w[lane] = ti - t;
    }
    __syncthreads();
    double run = s_w[wp] + inc - tot;
    for (int i = b; i < e; ++i) { run += src(i); dst[i] = run; }
    __syncthreads();
}

struct FieldStaticArgs {
    const double* rho;
    double *phi, *E;
    float* E32;     // may be null
    double* S;      // scratch: N doubles, every one written by scan 1 before anything reads it
    double* Tt;     // scratch: N doubles, every one written by scan 2 before anything reads it
    int N, nodes, bc;
    double phi0;
};

// One block.  S_j = sum_{i=1..j} (rho_i - mean), S_0 = 0; T_j = sum_{i=0..j} S_i; the closed form of the Thomas
// recurrences (L142), see the header.
__global__ void __launch_bounds__(1024) k_field_static(FieldStaticArgs a) {
    const int N = a.N, tid = threadIdx.x;
    const double* rho = a.rho;
    double mean = 0.0;
    if (a.bc == 1) {
        double p = 0.0;
        for (int i = tid; i < N; i += blockDim.x) p += rho[i];
        mean = fs_block_sum(p) / (double)N;
    }
    fs_block_scan([=](int i) { return i == 0 ? 0.0 : rho[i] - mean; }, a.S, N);
    const double* S = a.S;
    fs_block_scan([=](int i) { return S[i]; }, a.Tt, N);
    const double phi0 = a.bc == 0 ? a.phi0 : 0.0;
    const double phiN = 0.0;
    const double d1 = (phiN - phi0 + a.Tt[N - 1]) / (double)N;
    double psum = 0.0;
    for (int j = tid; j < a.nodes; j += blockDim.x) {
        double phi, E;
        if (j == 0) {
            phi = phi0;
            E = a.bc == 0 ? -d1 - rho[0] : -d1 + 0.5 * S[N - 1];  // bounded: half-cell Gauss law at the wall
        } else if (j == N) {                                        // bounded only: the right wall
            phi = phiN;
            E = -d1 + S[N - 1] + rho[N];
        } else {
            phi = phi0 + (double)j * d1 - a.Tt[j - 1];
            E = -d1 + 0.5 * (S[j - 1] + S[j]);
        }
        a.phi[j] = phi;
        a.E[j] = E;
        if (a.E32) a.E32[j] = (float)E;
        psum += phi;
    }
    if (a.bc == 1) {  // periodic: phi is defined up to a constant; report it with zero mean
        const double pm = fs_block_sum(psum) / (double)N;
        for (int j = tid; j < N; j += blockDim.x) a.phi[j] -= pm;  // each thread rewrites only its own nodes
    }
}

// ---- host side -------------------------------------------------------------------------------------------
constexpr int FS_MAX_DEVICES = 64;
std::mutex g_mu;
double* g_scratch_dev[FS_MAX_DEVICES];  // device address of g_field_scratch on device d, null = not looked up yet
thread_local char t_err[256] = "";

int fs_fail(int code, const char* fmt, ...) __attribute__((format(printf, 2, 3)));
int fs_fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
    return code;
}

// Device address of the scratch array on the CURRENT device.  The first call per device asks the runtime
// (cudaGetSymbolAddress resolves the symbol for the device that is current when it is called); the answer never
// changes afterwards, so it is cached per device ordinal.
int fs_scratch(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess)
        return fs_fail(PIC1D_ERR_CUDA, "pic1d_field_solve_static: cudaGetDevice failed: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= FS_MAX_DEVICES)
        return fs_fail(PIC1D_ERR_CUDA, "pic1d_field_solve_static: device ordinal %d is outside 0..%d", dev, FS_MAX_DEVICES - 1);
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_scratch_dev[dev] == nullptr) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_field_scratch);
        if (e != cudaSuccess || p == nullptr)
            return fs_fail(PIC1D_ERR_CUDA, "pic1d_field_solve_static: cudaGetSymbolAddress(scratch) failed on device %d: %s",
                           dev, cudaGetErrorString(e));
        g_scratch_dev[dev] = static_cast<double*>(p);
    }
    *out = g_scratch_dev[dev];
    return PIC1D_OK;
}

}  // namespace

extern "C" int pic1d_field_solve_static(const double* rho, double* phi, double* E, float* E32, int n_cells, int bc,
                                        double phi0, void* cuda_stream) {
    if (n_cells > PIC1D_FIELD_STATIC_MAX_CELLS)
        return fs_fail(PIC1D_ERR_ARG,
                       "pic1d_field_solve_static: n_cells = %d exceeds the built-in scratch array (at most %d cells); "
                       "use pic1d_create with a caller-allocated workspace for larger grids",
                       n_cells, PIC1D_FIELD_STATIC_MAX_CELLS);
    if (n_cells < 2) return fs_fail(PIC1D_ERR_ARG, "pic1d_field_solve_static: n_cells = %d, need at least 2", n_cells);
    if (bc != 0 && bc != 1) return fs_fail(PIC1D_ERR_ARG, "pic1d_field_solve_static: bc = %d, need 0 (bounded) or 1 (periodic)", bc);
    if (rho == nullptr || phi == nullptr || E == nullptr)
        return fs_fail(PIC1D_ERR_ARG, "pic1d_field_solve_static: rho, phi and E must be device pointers, not NULL");
    if (!std::isfinite(phi0)) return fs_fail(PIC1D_ERR_ARG, "pic1d_field_solve_static: phi0 is not finite");
    double* scratch = nullptr;
    const int rc = fs_scratch(&scratch);
    if (rc != PIC1D_OK) return rc;
    FieldStaticArgs a;
    a.rho = rho; a.phi = phi; a.E = E; a.E32 = E32;
    a.S = scratch;                                   // the looked-up DEVICE address, never the host-side symbol
    a.Tt = scratch + PIC1D_FIELD_STATIC_MAX_CELLS;
    a.N = n_cells; a.nodes = bc == 0 ? n_cells + 1 : n_cells; a.bc = bc; a.phi0 = phi0;
    k_field_static<<<1, 1024, 0, static_cast<cudaStream_t>(cuda_stream)>>>(a);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess)
        return fs_fail(PIC1D_ERR_CUDA, "pic1d_field_solve_static: kernel launch failed: %s", cudaGetErrorString(e));
    return PIC1D_OK;
}

extern "C" const char* pic1d_field_solve_static_error(void) { return t_err; }
