// pic1d_device.cuh -- device-side state and small device helpers (sm_100a).
//
// Compiled with -fmad=false: every fp32 operation is the IEEE operation that is written; fused
// multiply-adds appear only as explicit __fmaf_rn.  No fast-math, IEEE div / sqrt.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#define PIC1D_NT 256          // threads per block of the particle kernels
#define PIC1D_NWARP (PIC1D_NT / 32)
#define PIC1D_WA_MAX 1920     // bins of a tile window ranked at a time in shared memory (multiple of 8)
#define PIC1D_GROUP 64        // tiles per tile-group (window union used by the bin scan)
#define PIC1D_DEAD_CHUNKS 64  // blocks that scan the per-tile absorbed counts (see DevSpecies)

// Philox stream ids (R12)
#define STREAM_NULL 0u
#define STREAM_COLL 2u
#define STREAM_SEE 4u
#define STREAM_REFL 5u  // electron reflection at the walls (f4)
#define STREAM_COUL 6u  // + species: binary Coulomb collisions inside sort cells (f3)

// sticky error bits in DevState::err
#define ERRBIT_CAPACITY 1u
#define ERRBIT_NONFINITE 2u
#define ERRBIT_WORKSPACE 4u
#define ERRBIT_BADLOAD 8u

typedef unsigned long long ull;

// Per-species device-resident scalars.  Everything a step needs to know about particle counts
// lives here, so a step never synchronises with the host.
struct DevSpecies {
    int n_live;    // N_s: live slots in the current buffer (sorted part + birth tail)
    int n_sorted;  // sorted part
    int n_push;    // slots [0, n_push) are pushed by the running sort; [n_push, n_src) are not
    int n_src;     // source slots of the running sort (n_push + injected secondaries)
    int n_tiles;   // ceil(n_src / T) of the running sort
    int n_dead;    // absorbed particles of the running sort
    int pool_used; // entries of the (tile x bin) count pool in use
    int ticket;    // dynamic tile counter of the MCC kernel
    int ticket2;   // dynamic tile counter of the scatter kernel
    int scan_done; // bin blocks of k_bin_scan that have finished (the last one scans the histogram)
    ull absorbed_left, absorbed_right, injected, n_candidates, n_events[4], births, dropped, over_cap;
    ull reflected, n_pairs;  // f4: electrons reflected at a wall; f3: binary collisions performed
    // ordered absorbed list (ions with secondary emission): the per-tile absorbed counts are scanned in
    // PIC1D_DEAD_CHUNKS chunks by as many blocks; the block that finishes last turns the chunk totals into bases
    int dead_done;
    int dead_tot[PIC1D_DEAD_CHUNKS], dead_base[PIC1D_DEAD_CHUNKS];
};

struct DevState {
    DevSpecies sp[2];
    unsigned int step;       // n: index of the step being computed (set by k_step_begin)
    unsigned int err;        // sticky ERRBIT_*
    int n_abs;               // absorbed ions recorded in the list this step
    unsigned int step_next;  // index the next step will get
};

// Philox4x32-10 (Salmon et al., SC'11).  key = (seed_lo, seed_hi).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// U(r) = (r >> 8) * 2^-24 in [0, 1), exact in fp32
__device__ __forceinline__ float u01(uint32_t r) { return __fmul_rn((float)(r >> 8), 0x1p-24f); }

__device__ __forceinline__ unsigned lanemask_lt() {
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// shared-memory fetch-and-add issued by ONE lane that already carries a warp-aggregated value: plain
// atom.shared, so that ptxas does not wrap it in its own (20-instruction) warp-aggregation sequence
__device__ __forceinline__ int atom_shared_add(int* p, int v) {
    int old;
    const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(a), "r"(v) : "memory");
    return old;
}

// tiles per chunk of the absorbed-count scan (a multiple of 32); the same on both sides of the scan
__device__ __forceinline__ int dead_chunk_tiles(int n_tiles) {
    return ((n_tiles + PIC1D_DEAD_CHUNKS - 1) / PIC1D_DEAD_CHUNKS + 31) & ~31;
}

__device__ __forceinline__ int warp_min(int v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ int warp_max(int v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ int warp_sum(int v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// f4, electron reflection at the walls (L41; R22): prob = 0 switches it off
struct ReflP {
    float prob;
    uint32_t k0, k1;
};

// Gather + leapfrog push + boundary + sort key for ONE particle (PAPER.md L35, L87, L150-156,
// Eq. 3-4; boundary L41; key L63-67).  Used verbatim by the counting pass and by the scatter pass,
// so both see bit-identical x, vx and key.  slot = the particle's source slot (keys the reflection draw);
// n_refl counts the reflections.
//   key >= 0 : sort cell;  -1 : absorbed at the left wall;  -2 : absorbed at the right wall / NaN
template <int BC>
__device__ __forceinline__ int push_particle(float& x, float& vx, bool do_push,
                                             const float* __restrict__ E32, float kappa, int Nc,
                                             float fNc, float inv_r, int shift,
                                             const ReflP& rp, uint32_t step, unsigned slot, int& n_refl) {
    if (do_push) {
        int j = (int)x;  // "single type casting operation", L87
        float f = __fsub_rn(x, (float)j);
        int j1 = j + 1;
        if (BC == 1 && j1 == Nc) j1 = 0;
        float e0 = __ldg(E32 + j), e1 = __ldg(E32 + j1);
        float Ep = __fmaf_rn(f, __fsub_rn(e1, e0), e0);
        vx = __fmaf_rn(kappa, Ep, vx);  // v(t+1/2) = v(t-1/2) + kappa E(x(t))   L152
        x = __fadd_rn(x, vx);           // x(t+1) = x(t) + v(t+1/2)              L154
    }
    if (BC == 1) {
        if (x < 0.0f) x = __fadd_rn(x, fNc);
        if (x >= fNc) x = __fsub_rn(x, fNc);
        if (!(x >= 0.0f && x < fNc)) x = 0.0f;  // rounding of -tiny + N_c, |v| > N_c, non-finite
    } else if (!(x >= 0.0f && x < fNc)) {
        bool back = false;
        if (rp.prob > 0.0f && do_push && x == x) {  // with probability prob: mirror position, vx reversed
            uint32_t w[4];
            philox4x32_10(slot, step, STREAM_REFL, 0u, rp.k0, rp.k1, w);
            if (u01(w[0]) < rp.prob) {
                const float xr = x < 0.0f ? -x : __fsub_rn(__fmul_rn(2.0f, fNc), x);
                if (xr >= 0.0f && xr < fNc) { x = xr; vx = -vx; back = true; ++n_refl; }
            }
        }
        if (!back) return x < 0.0f ? -1 : -2;
    }
    return ((int)__fmul_rn(x, inv_r)) >> shift;  // shift > 0 only in the coarse pass of a load
}
