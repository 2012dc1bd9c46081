// pic1d_gsort.cu -- the paper's gapped in-place fine sort fused with the pusher (include/pic1d_gsort.h;
// PAPER.md L160-192, Fig. 6-9), one thread block per sort cell as in the paper (L67, Fig. 3).
//
// What is kept of the paper's design: fixed-capacity cells with the free slots as sorting buffer, rejected
// particles to the END of the cell through a shared counter (1a), gaps closed from the end (1b), neighbours'
// rejected buffers only READ in step 2, a global atomic counter only for the rare far movers of step 3.
// What differs on a B200: SoA arrays instead of float4 AoS (the in-place push then touches only x and vx:
// 16 B per particle-step), every thread remembers its own rejected slots in a register bit mask (no flags in
// memory), and particles that left the box are dropped right in kernel 1 (they need no buffer slot).
#include <cmath>
#include <new>

#include "../../include/pic1d.h"
#include "../../include/pic1d_gsort.h"
#include "pic1d_device.cuh"

namespace {

#define GS_NT 256
#define GS_PT 32  // particles per thread and cell at most: n_max <= GS_NT * GS_PT = 8192
#define GS_U 8    // of them in flight together

struct GsState {
    ull absorbed_left, absorbed_right, moved_near, moved_far;
    unsigned err;
    unsigned pad;
};

struct GsArgs {
    float *x, *vx, *vy, *vz;
    int *N, *R;
    const float* E32;
    GsState* st;
    int n_cells, n_sc, n_max;
    float inv_r, kappa, fNc;
};

// kernel 1: push in place + step 1a + step 1b
__global__ void __launch_bounds__(GS_NT) k_gs_push(GsArgs a) {
    extern __shared__ unsigned short s_hole[];  // [n_max] positions of the gaps below the new valid count
    __shared__ int s_top, s_holes, s_nh, s_nd, s_abs[2];
    const int tid = threadIdx.x;
    const ReflP norefl = {0.0f, 0u, 0u};
    for (int c = blockIdx.x; c < a.n_sc; c += gridDim.x) {
        const size_t base = (size_t)c * a.n_max;
        const int N = a.N[c];
        if (tid == 0) { s_top = a.n_max; s_holes = 0; s_nh = 0; s_nd = 0; s_abs[0] = 0; s_abs[1] = 0; }
        __syncthreads();
        unsigned rej = 0;  // bit it: my particle tid + it * GS_NT left the cell
        // GS_U particles per thread at a time: their loads are independent and in flight together (a thread's own
        // slots j < N are read before anything is written to them; rejected particles go to slots >= N)
        for (int it0 = 0; it0 < GS_PT && it0 * GS_NT < N; it0 += GS_U) {
            float xs[GS_U], vs[GS_U];
#pragma unroll
            for (int u = 0; u < GS_U; ++u) {
                const int j = tid + (it0 + u) * GS_NT;
                xs[u] = 0.0f; vs[u] = 0.0f;
                if (j < N) { xs[u] = __ldcs(a.x + base + j); vs[u] = __ldcs(a.vx + base + j); }
            }
#pragma unroll
            for (int u = 0; u < GS_U; ++u) {
                const int it = it0 + u, j = tid + it * GS_NT;
                if (j >= N) continue;
                float x = xs[u], vx = vs[u];
                int dummy = 0;
                const int key = push_particle<0>(x, vx, true, a.E32, a.kappa, a.n_cells, a.fNc, a.inv_r, 0, norefl, 0u, 0u, dummy);
                a.x[base + j] = x; a.vx[base + j] = vx;  // in place, whether it stays or not
                if (key != c) rej |= 1u << it;           // the rare path is taken after the loop
            }
        }
        // step 1a for the thread's rejected particles (few): to the end of the cell through the shared counter
        if (rej) atomicAdd(&s_holes, __popc(rej));
        for (unsigned todo = rej; todo; todo &= todo - 1u) {
            const int j = tid + (__ffs(todo) - 1) * GS_NT;
            const float x = a.x[base + j];  // this thread's own store above
            if (!(x >= 0.0f && x < a.fNc)) { atomicAdd(&s_abs[x < 0.0f ? 0 : 1], 1); continue; }  // left the box (L41): dropped
            const int idx = atomicSub(&s_top, 1) - 1;  // N_index counts down from the end of the cell
            if (idx < N) { atomicOr(&a.st->err, 1u); continue; }  // no free slot left: dropped, sticky error
            a.x[base + idx] = x; a.vx[base + idx] = a.vx[base + j];
            a.vy[base + idx] = a.vy[base + j]; a.vz[base + idx] = a.vz[base + j];
        }
        __syncthreads();
        const int V = N - s_holes;
        // step 1b: the gaps below V are closed with the valid particles at and above V
        for (int it = 0; it < GS_PT; ++it) {
            const int j = tid + it * GS_NT;
            if (j >= V) break;
            if ((rej >> it) & 1u) s_hole[atomicAdd(&s_nh, 1)] = (unsigned short)j;
        }
        __syncthreads();
        for (int it = 0; it < GS_PT; ++it) {
            const int j = tid + it * GS_NT;
            if (j >= N) break;
            if (j < V || ((rej >> it) & 1u)) continue;
            const int dst = s_hole[atomicAdd(&s_nd, 1)];
            a.x[base + dst] = a.x[base + j]; a.vx[base + dst] = a.vx[base + j];
            a.vy[base + dst] = a.vy[base + j]; a.vz[base + dst] = a.vz[base + j];
        }
        if (tid == 0) {
            a.N[c] = V;
            a.R[c] = a.n_max - max(s_top, N);
            if (s_abs[0]) atomicAdd(&a.st->absorbed_left, (ull)s_abs[0]);
            if (s_abs[1]) atomicAdd(&a.st->absorbed_right, (ull)s_abs[1]);
        }
        __syncthreads();
    }
}

__device__ __forceinline__ int gs_key(const GsArgs& a, float x) { return (int)__fmul_rn(x, a.inv_r); }

__device__ __forceinline__ void gs_copy(const GsArgs& a, size_t dst, size_t src) {
    a.x[dst] = a.x[src]; a.vx[dst] = a.vx[src]; a.vy[dst] = a.vy[src]; a.vz[dst] = a.vz[src];
}

// kernel 2: cell c takes what its neighbours rejected and belongs to c (the neighbours' buffers are only read)
__global__ void __launch_bounds__(GS_NT) k_gs_near(GsArgs a) {
    __shared__ int s_n;
    const int tid = threadIdx.x;
    for (int c = blockIdx.x; c < a.n_sc; c += gridDim.x) {
        const size_t base = (size_t)c * a.n_max;
        const int V = a.N[c], room = a.n_max - a.R[c] - V;
        if (tid == 0) s_n = 0;
        __syncthreads();
        for (int side = 0; side < 2; ++side) {
            const int nb = side == 0 ? c - 1 : c + 1;
            if (nb < 0 || nb >= a.n_sc) continue;
            const int Rn = a.R[nb];
            const size_t nbase = (size_t)nb * a.n_max + (size_t)(a.n_max - Rn);
            for (int q = tid; q < Rn; q += GS_NT) {
                if (gs_key(a, a.x[nbase + q]) != c) continue;
                const int idx = atomicAdd(&s_n, 1);
                if (idx < room) gs_copy(a, base + V + idx, nbase + q);
            }
        }
        __syncthreads();
        if (tid == 0) {
            const int got = s_n;
            if (got > room) atomicOr(&a.st->err, 1u);
            a.N[c] = V + min(got, room);
            if (got) atomicAdd(&a.st->moved_near, (ull)min(got, room));
        }
        __syncthreads();
    }
}

// kernel 3: rejected particles that moved farther than one cell; the sole global atomic index counter (L186)
__global__ void __launch_bounds__(GS_NT) k_gs_far(GsArgs a) {
    const int tid = threadIdx.x;
    for (int c = blockIdx.x; c < a.n_sc; c += gridDim.x) {
        const int Rc = a.R[c];
        const size_t rbase = (size_t)c * a.n_max + (size_t)(a.n_max - Rc);
        for (int q = tid; q < Rc; q += GS_NT) {
            const int k = gs_key(a, a.x[rbase + q]);
            if (k == c - 1 || k == c + 1) continue;
            const int idx = atomicAdd(&a.N[k], 1);
            if (idx < a.n_max - a.R[k]) {
                gs_copy(a, (size_t)k * a.n_max + idx, rbase + q);
                atomicAdd(&a.st->moved_far, 1ull);
            } else {
                atomicSub(&a.N[k], 1);
                atomicOr(&a.st->err, 1u);
            }
        }
    }
}

__global__ void k_gs_load(GsArgs a, const float* x, const float* vx, const float* vy, const float* vz, int n) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float xv = x[i];
        if (!(xv >= 0.0f && xv < a.fNc)) { atomicOr(&a.st->err, 2u); continue; }
        const int k = gs_key(a, xv);
        const int idx = atomicAdd(&a.N[k], 1);
        if (idx >= a.n_max) { atomicSub(&a.N[k], 1); atomicOr(&a.st->err, 1u); continue; }
        const size_t d = (size_t)k * a.n_max + idx;
        a.x[d] = xv; a.vx[d] = vx[i]; a.vy[d] = vy[i]; a.vz[d] = vz[i];
    }
}

inline size_t gs_align(size_t v) { return (v + 255) / 256 * 256; }

}  // namespace

struct pic1d_gsort {
    GsArgs a;
    cudaStream_t stream;
    float* stage[4];   // device staging of a host load
    size_t stage_cap;
    int num_sms;
    float* E32;
};

namespace {

size_t gs_layout(pic1d_gsort* h, char* base, int n_cells, double inv_ratio, int n_max) {
    GsArgs& a = h->a;
    a.n_cells = n_cells; a.n_max = n_max; a.inv_r = (float)inv_ratio; a.fNc = (float)n_cells;
    a.n_sc = (int)std::ceil((double)n_cells * inv_ratio);
    const size_t tot = (size_t)a.n_sc * (size_t)n_max;
    size_t off = 0;
    auto carve = [&](size_t bytes) { char* p = base ? base + off : nullptr; off = gs_align(off + bytes); return p; };
    a.st = reinterpret_cast<GsState*>(carve(sizeof(GsState)));
    a.x = reinterpret_cast<float*>(carve(tot * 4)); a.vx = reinterpret_cast<float*>(carve(tot * 4));
    a.vy = reinterpret_cast<float*>(carve(tot * 4)); a.vz = reinterpret_cast<float*>(carve(tot * 4));
    a.N = reinterpret_cast<int*>(carve((size_t)a.n_sc * 4)); a.R = reinterpret_cast<int*>(carve((size_t)a.n_sc * 4));
    h->E32 = reinterpret_cast<float*>(carve((size_t)(n_cells + 1) * 4));
    a.E32 = h->E32;
    h->stage_cap = tot;  // a host load is staged through the workspace
    for (int k = 0; k < 4; ++k) h->stage[k] = reinterpret_cast<float*>(carve(tot * 4));
    return off;
}

int gs_check(int n_cells, double inv_ratio, int n_max) {
    if (n_cells < 2 || n_cells > (1 << 24) || n_max < 1 || n_max > GS_NT * GS_PT || !(inv_ratio > 0.0)) return PIC1D_ERR_ARG;
    int e;
    if (std::frexp(inv_ratio, &e) != 0.5) return PIC1D_ERR_ARG;
    return PIC1D_OK;
}

}  // namespace

extern "C" {

int pic1d_gsort_workspace_bytes(int n_cells, double sort_inv_ratio, int n_max, size_t* bytes_out) {
    if (!bytes_out || gs_check(n_cells, sort_inv_ratio, n_max)) return PIC1D_ERR_ARG;
    pic1d_gsort tmp{};
    *bytes_out = gs_layout(&tmp, nullptr, n_cells, sort_inv_ratio, n_max);
    return PIC1D_OK;
}

int pic1d_gsort_create(int n_cells, double sort_inv_ratio, int n_max, double kappa, void* workspace,
                       size_t workspace_bytes, void* cuda_stream, pic1d_gsort_t** out) {
    if (!out || !workspace || gs_check(n_cells, sort_inv_ratio, n_max)) return PIC1D_ERR_ARG;
    if (reinterpret_cast<uintptr_t>(workspace) % 256 != 0) return PIC1D_ERR_ARG;
    pic1d_gsort* h = new (std::nothrow) pic1d_gsort{};
    if (!h) return PIC1D_ERR_ARG;
    if (gs_layout(h, reinterpret_cast<char*>(workspace), n_cells, sort_inv_ratio, n_max) > workspace_bytes) {
        delete h;
        return PIC1D_ERR_WORKSPACE;
    }
    h->a.kappa = (float)kappa;
    h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { delete h; return PIC1D_ERR_CUDA; }
    h->num_sms = prop.multiProcessorCount;
    cudaMemsetAsync(h->a.st, 0, sizeof(GsState), h->stream);
    cudaMemsetAsync(h->a.N, 0, sizeof(int) * h->a.n_sc, h->stream);
    cudaMemsetAsync(h->a.R, 0, sizeof(int) * h->a.n_sc, h->stream);
    cudaMemsetAsync(h->E32, 0, sizeof(float) * (n_cells + 1), h->stream);
    if (cudaGetLastError() != cudaSuccess) { delete h; return PIC1D_ERR_CUDA; }
    *out = h;
    return PIC1D_OK;
}

int pic1d_gsort_load(pic1d_gsort_t* h, int64_t n, const float* x, const float* vx, const float* vy,
                     const float* vz, int on_device) {
    if (!h || n < 0 || (n > 0 && (!x || !vx || !vy || !vz))) return PIC1D_ERR_ARG;
    if (!on_device && (size_t)n > h->stage_cap) return PIC1D_ERR_CAPACITY;
    cudaMemsetAsync(h->a.st, 0, sizeof(GsState), h->stream);
    cudaMemsetAsync(h->a.N, 0, sizeof(int) * h->a.n_sc, h->stream);
    cudaMemsetAsync(h->a.R, 0, sizeof(int) * h->a.n_sc, h->stream);
    const float* src[4] = {x, vx, vy, vz};
    if (!on_device) {
        for (int k = 0; k < 4 && n > 0; ++k) {
            if (cudaMemcpyAsync(h->stage[k], src[k], (size_t)n * 4, cudaMemcpyHostToDevice, h->stream) != cudaSuccess) return PIC1D_ERR_CUDA;
            src[k] = h->stage[k];
        }
    }
    if (n > 0) k_gs_load<<<(int)std::min<int64_t>((n + 255) / 256, h->num_sms * 8), 256, 0, h->stream>>>(h->a, src[0], src[1], src[2], src[3], (int)n);
    if (cudaGetLastError() != cudaSuccess) return PIC1D_ERR_CUDA;
    if (!on_device && cudaStreamSynchronize(h->stream) != cudaSuccess) return PIC1D_ERR_CUDA;
    return PIC1D_OK;
}

int pic1d_gsort_set_E32(pic1d_gsort_t* h, const float* E32, int n_nodes, int on_device) {
    if (!h || !E32 || n_nodes != h->a.n_cells + 1) return PIC1D_ERR_ARG;
    if (cudaMemcpyAsync(h->E32, E32, sizeof(float) * n_nodes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice,
                        h->stream) != cudaSuccess) return PIC1D_ERR_CUDA;
    if (!on_device && cudaStreamSynchronize(h->stream) != cudaSuccess) return PIC1D_ERR_CUDA;
    return PIC1D_OK;
}

int pic1d_gsort_step(pic1d_gsort_t* h, int n_steps) {
    if (!h || n_steps < 0) return PIC1D_ERR_ARG;
    const int grid = std::min(h->a.n_sc, h->num_sms * 8);
    for (int s = 0; s < n_steps; ++s) {
        k_gs_push<<<grid, GS_NT, (size_t)h->a.n_max * sizeof(unsigned short), h->stream>>>(h->a);
        k_gs_near<<<grid, GS_NT, 0, h->stream>>>(h->a);
        k_gs_far<<<grid, GS_NT, 0, h->stream>>>(h->a);
    }
    return cudaGetLastError() == cudaSuccess ? PIC1D_OK : PIC1D_ERR_CUDA;
}

int pic1d_gsort_get(pic1d_gsort_t* h, int32_t* N_i, float* x, float* vx, float* vy, float* vz, int64_t* stats) {
    if (!h) return PIC1D_ERR_ARG;
    const size_t tot = (size_t)h->a.n_sc * (size_t)h->a.n_max;
    GsState st;
    bool ok = cudaMemcpyAsync(&st, h->a.st, sizeof(st), cudaMemcpyDeviceToHost, h->stream) == cudaSuccess;
    if (N_i) ok = ok && cudaMemcpyAsync(N_i, h->a.N, sizeof(int) * h->a.n_sc, cudaMemcpyDeviceToHost, h->stream) == cudaSuccess;
    float* dst[4] = {x, vx, vy, vz};
    const float* src[4] = {h->a.x, h->a.vx, h->a.vy, h->a.vz};
    for (int k = 0; k < 4; ++k)
        if (dst[k]) ok = ok && cudaMemcpyAsync(dst[k], src[k], tot * 4, cudaMemcpyDeviceToHost, h->stream) == cudaSuccess;
    if (!ok || cudaStreamSynchronize(h->stream) != cudaSuccess) return PIC1D_ERR_CUDA;
    const int sticky = (st.err & 1u) ? PIC1D_ERR_CAPACITY : ((st.err & 2u) ? PIC1D_ERR_ARG : PIC1D_OK);
    if (stats) {
        stats[0] = (int64_t)st.absorbed_left; stats[1] = (int64_t)st.absorbed_right;
        stats[2] = (int64_t)st.moved_near; stats[3] = (int64_t)st.moved_far; stats[4] = sticky;
    }
    return sticky;
}

int pic1d_gsort_n_sort_cells(const pic1d_gsort_t* h) { return h ? h->a.n_sc : PIC1D_ERR_ARG; }

int pic1d_gsort_destroy(pic1d_gsort_t* h) {
    if (!h) return PIC1D_OK;
    cudaStreamSynchronize(h->stream);
    delete h;
    return PIC1D_OK;
}

}  // extern "C"
