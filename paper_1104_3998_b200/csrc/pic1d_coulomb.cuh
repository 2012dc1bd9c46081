// pic1d_coulomb.cuh -- binary Coulomb collisions inside sort cells.
//
// The paper names them as THE reason for fine sorting ("allows for a straightforward and fast implementation
// of nonlinear collision processes (i.e. Coulomb collisions) through the binary collisions"; L75,
// L221, L259) but does not implement them.  The sorted per-cell ranges offsets[k] .. offsets[k+1] built by the
// fine sort are exactly the data structure the binary-collision model of Takizuka & Abe (J. Comput. Phys. 25
// (1977) 205) needs: the n particles of a sort cell are paired, a pair with relative velocity u is scattered by
// theta with tan(theta/2) = delta ~ N(0, coul_A n / u^3) and a uniform azimuth, each partner takes half of the
// change of u (like particles: equal mass and weight), so momentum and energy of every pair are conserved.
// Pairing (R23): a keyed pseudo-random permutation pi of the cell's sorted slots -- four balanced Feistel
// rounds on 2h bits (4^h >= n) keyed by philox(cell, step, COUL + s, 0), cycle-walked into [0, n) -- so that any
// pairing of the cell can come out; pairs (pi(2m), pi(2m+1)); for odd n slot pi(n-1) sits out (not Takizuka-Abe's
// three-particle rule).  Every thread evaluates pi for its own pairs: integer work, bit-identical to the oracle's.
// One block per sort cell, one thread per pair; the cell's velocities (12 B x n) are staged in shared memory.
// fp32 operations in the order the oracle states them (-fmad=false: nothing is contracted).
#pragma once
#include "pic1d_device.cuh"
#include "pic1d_mcc.cuh"

struct CoulombArgs {
    float *vx, *vy, *vz;   // the species' sorted buffer
    const int* offsets;    // [n_sc + 1]
    int* partner;          // optional (PIC1D_FLAG_CAPTURE): partner slot per sorted slot, -1 = sits out
    DevState* st;
    int s, n_sc;
    float A;               // coul_A
    uint32_t k0, k1;
    int slots;             // particles per cell the shared-memory staging holds (dynamic smem = 12 B x slots)
};

__device__ __forceinline__ unsigned coul_feistel(unsigned m, unsigned n, unsigned h, const uint32_t (&w)[4]) {
    const unsigned mask = (1u << h) - 1u;
    unsigned x = m;
    do {  // cycle walking: a cycle of the permutation of [0, 4^h) that starts below n returns below n
        unsigned L = x >> h, R = x & mask;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            unsigned z = (R ^ w[r]) * 0x9E3779B1u;
            z ^= z >> 15; z *= 0x85EBCA77u; z ^= z >> 13;
            const unsigned t = L ^ (z & mask);
            L = R; R = t;
        }
        x = (L << h) | R;
    } while (x >= n);
    return x;
}

// One pair: the oracle's operation order, on values read from / written to `vx, vy, vz` at ia, ib (global arrays
// with global slots, or the cell's shared-memory copy with slots relative to the cell).  `key` = the pair's first
// GLOBAL slot (the Philox counter).
__device__ __forceinline__ void coul_pair(float* vx, float* vy, float* vz, unsigned ia, unsigned ib, unsigned key,
                                          uint32_t step, uint32_t stream, const CoulombArgs& a, float fn) {
    const float vxa = vx[ia], vya = vy[ia], vza = vz[ia];
    const float vxb = vx[ib], vyb = vy[ib], vzb = vz[ib];
    const float ux = vxa - vxb, uy = vya - vyb, uz = vza - vzb;
    const float up2 = ux * ux + uy * uy;
    const float u2 = up2 + uz * uz;
    if (!(u2 > 0.0f)) return;
    uint32_t r[4];
    philox4x32_10(key, step, stream, 1u, a.k0, a.k1, r);  // keyed on the pair's first slot
    const float uu = sqrtf(u2), up = sqrtf(up2);
    const float var = (a.A * fn) / (u2 * uu);
    const float delta = sqrtf(var) * (bm_r(u01(r[0])) * cosf(6.2831855f * u01(r[1])));
    const float d2 = delta * delta;
    const float sint = (2.0f * delta) / (1.0f + d2);
    const float omc = (2.0f * d2) / (1.0f + d2);  // 1 - cos(theta)
    const float ph = 6.2831855f * u01(r[2]);
    const float cp = cosf(ph), sp = sinf(ph);
    float dux, duy, duz;
    if (up > 0.0f) {
        dux = ((ux / up) * uz) * (sint * cp) - ((uy / up) * uu) * (sint * sp) - ux * omc;
        duy = ((uy / up) * uz) * (sint * cp) + ((ux / up) * uu) * (sint * sp) - uy * omc;
        duz = -(up * (sint * cp)) - uz * omc;
    } else {
        dux = uu * (sint * cp); duy = uu * (sint * sp); duz = -(uz * omc);
    }
    vx[ia] = vxa + 0.5f * dux; vy[ia] = vya + 0.5f * duy; vz[ia] = vza + 0.5f * duz;
    vx[ib] = vxb - 0.5f * dux; vy[ib] = vyb - 0.5f * duy; vz[ib] = vzb - 0.5f * duz;
}

// A cell of up to a.slots particles is staged: its three velocity arrays are read into shared memory with
// coalesced loads, the pairs (random slots of the cell) are scattered there, and the arrays are written back
// coalesced -- the partners' gathers cost shared-memory bank conflicts instead of one 32-byte sector per lane
// (measured on config 4: 29.6 sectors per request, 0.09 of the HBM peak before; profiles/r3_next_kernels.md).
// Larger cells take the gathered path.  Every particle is in at most one pair, so the order of the pairs does not
// matter and both paths give the bits of the oracle's sequential loop.
__global__ void __launch_bounds__(PIC1D_NT) k_coulomb(CoulombArgs a) {
    extern __shared__ float s_v[];  // [3 * a.slots]
    float* const s_vx = s_v;
    float* const s_vy = s_v + a.slots;
    float* const s_vz = s_v + 2 * a.slots;
    const int tid = threadIdx.x, lane = tid & 31;
    const uint32_t step = a.st->step;
    const uint32_t stream = STREAM_COUL + (uint32_t)a.s;
    unsigned n_pairs = 0;
    for (int k = blockIdx.x; k < a.n_sc; k += gridDim.x) {
        const unsigned off = (unsigned)a.offsets[k], n = (unsigned)(a.offsets[k + 1] - a.offsets[k]);
        if (n < 2u) {
            if (a.partner && n == 1u && tid == 0) a.partner[off] = -1;
            continue;
        }
        uint32_t w[4];
        philox4x32_10((uint32_t)k, step, stream, 0u, a.k0, a.k1, w);  // every thread: the cell's permutation
        unsigned h = 1u;
        while ((1ull << (2u * h)) < n) ++h;  // 4^h >= n
        const float fn = (float)n;
        if (a.partner && (n & 1u) && tid == 0) a.partner[off + coul_feistel(n - 1u, n, h, w)] = -1;
        const bool staged = n <= (unsigned)a.slots;  // block-uniform
        if (staged) {
            for (unsigned i = tid; i < n; i += PIC1D_NT) {
                s_vx[i] = a.vx[off + i]; s_vy[i] = a.vy[off + i]; s_vz[i] = a.vz[off + i];
            }
            __syncthreads();
        }
        for (unsigned m = 2u * tid; m + 1u < n; m += 2u * PIC1D_NT) {
            const unsigned ia = coul_feistel(m, n, h, w), ib = coul_feistel(m + 1u, n, h, w);
            if (a.partner) { a.partner[off + ia] = (int)(off + ib); a.partner[off + ib] = (int)(off + ia); }
            ++n_pairs;
            if (staged) coul_pair(s_vx, s_vy, s_vz, ia, ib, off + ia, step, stream, a, fn);
            else coul_pair(a.vx, a.vy, a.vz, off + ia, off + ib, off + ia, step, stream, a, fn);
        }
        if (staged) {
            __syncthreads();
            for (unsigned i = tid; i < n; i += PIC1D_NT) {
                a.vx[off + i] = s_vx[i]; a.vy[off + i] = s_vy[i]; a.vz[off + i] = s_vz[i];
            }
            __syncthreads();  // the next cell overwrites the staging arrays
        }
    }
    n_pairs = __reduce_add_sync(0xffffffffu, n_pairs);
    if (lane == 0 && n_pairs) atomicAdd(&a.st->sp[a.s].n_pairs, (ull)n_pairs);
}
