// pic1d_mcc.cuh -- modified null-collision Monte-Carlo collisions (Eq. 6).
//
// Every sorted particle draws p (L203); p < P0 enters the standard null-collision selection with the
// synthetic analytic cross sections (products and sums only, in the spirit of L207).  The paper notes
// that this module has "lots of branches" (L209); here the branches are removed by compaction inside
// a tile of MCC_TILE sorted slots:
//   phase A  null test for every slot: one Philox call serves 4 consecutive slots (R12);
//            nothing is loaded; candidates are compacted into a shared list
//   phase B  one thread per CANDIDATE: load v, Philox (u_type, ...), process selection (no
//            transcendental); real collisions are compacted into a second list
//   phase C  one thread per REAL COLLISION: kinematics (sqrt, sincos, log), velocity written back
//   k_mcc_births  one thread per IONISATION: the new electron / ion pair
// Ionisation products go to the tails of the electron / ion arrays in ascending parent-slot order
// (the paper allocates them with a shared counter inside the parent's sort cell, L203; here the tail
// is sorted into place by the next step's fine sort).  The order inside a tile comes from a bit mask
// over its slots, the order across tiles from the prefix of the per-tile ionisation counts that
// k_mcc_births forms -- no atomic decides any index.
#pragma once
#include "pic1d_device.cuh"

#define MCC_TILE (PIC1D_NT * 16)       // sorted slots per tile
#define MCC_TILE_STAGE (PIC1D_NT * 16) // ... when the velocities are staged in shared memory (8: slower)

struct MccArgs {
    float *x, *vx, *vy, *vz;      // this species' current (sorted) buffer
    float *ex, *evx, *evy, *evz;  // electron buffer (birth tail)
    float *ix, *ivx, *ivy, *ivz;  // ion buffer (birth tail), may be null
    DevState* st;
    int* rec_nb;     // [tile] ionisations of the tile (electron set)
    int* rec_rel;    // [tile * MCC_TILE + r] parent slot - tile base of the tile's r-th ionisation, slot order
    float* rec_gp;   // [tile * MCC_TILE + r] speed shared by its two electrons
    uint8_t* mask;   // optional event mask per sorted slot
    int s, kind, n_species, cap_e, cap_i;
    uint32_t step, k0, k1;
    uint32_t null_le;  // null test in integers: U(w) < P0  <=>  w <= null_le   (null_any = 0: never)
    int null_any;
    float P0, inv_g_cap, c_eV, r_el, r_exc, r_ion, E_exc, E_ion, two_mr, gvt;
};

__device__ __forceinline__ void iso_dir(float ua, float ub, float (&n)[3]) {
    const float ct = __fsub_rn(1.0f, __fmul_rn(2.0f, ua));
    const float st = sqrtf(fmaxf(0.0f, __fsub_rn(1.0f, __fmul_rn(ct, ct))));
    const float ph = __fmul_rn(6.2831855f, ub);
    n[0] = ct;
    n[1] = __fmul_rn(st, cosf(ph));
    n[2] = __fmul_rn(st, sinf(ph));
}
__device__ __forceinline__ float bm_r(float u) {
    return sqrtf(__fmul_rn(-2.0f, logf(__fsub_rn(1.0f, u))));
}

// append `flag`-ged items of a warp to a shared list; returns this lane's index (valid if flag)
__device__ __forceinline__ int warp_append(bool flag, int* counter) {
    const unsigned bal = __ballot_sync(0xffffffffu, flag);
    int base = 0;
    if ((threadIdx.x & 31) == 0 && bal) base = atom_shared_add(counter, __popc(bal));
    base = __shfl_sync(0xffffffffu, base, 0);
    return base + __popc(bal & lanemask_lt());
}

// KIND: 1 electron set, 2 ion charge exchange.  STAGE: phase A streams the tile's vx, vy, vz into shared
// memory with vector loads while it computes the null tests (worth it when most slots are candidates);
// otherwise phases B / C fetch the few candidates' velocities from global memory.
template <int KIND, bool STAGE>
__global__ void __launch_bounds__(PIC1D_NT, STAGE ? 3 : 4) k_mcc(MccArgs a) {
    constexpr int TILE = STAGE ? MCC_TILE_STAGE : MCC_TILE;
    extern __shared__ float s_v[];  // STAGE: [3][TILE] velocities
    __shared__ int s_tile;
    __shared__ int s_n[3];                          // candidates, real collisions, ionisations
    __shared__ unsigned short s_cand[TILE];     // slot - tile base
    __shared__ unsigned short s_coll[TILE];     // (slot - tile base) | event << 12
    __shared__ unsigned s_ionbits[TILE / 32];   // bit = slot ionises
    const int tid = threadIdx.x, lane = tid & 31;
    DevState* st = a.st;
    DevSpecies& sp = st->sp[a.s];
    const int n_sorted = sp.n_sorted;
    const int n_act = (n_sorted + TILE - 1) / TILE;
    const uint32_t str_null = STREAM_NULL + (uint32_t)a.s, str_coll = STREAM_COLL + (uint32_t)a.s;
    int c_cand = 0, c_e0 = 0, c_e1 = 0, c_e2 = 0, c_e3 = 0, c_over = 0;
    float* s_vx = s_v; float* s_vy = s_v + TILE; float* s_vz = s_v + 2 * TILE;
    while (true) {
        if (tid == 0) { s_tile = atomicAdd(&sp.ticket, 1); s_n[0] = 0; s_n[1] = 0; s_n[2] = 0; }
        if (tid < TILE / 32) s_ionbits[tid] = 0u;
        __syncthreads();
        const int tile = s_tile;
        if (tile >= n_act) break;
        const int tbase = tile * TILE;
        // ---- phase A: null test, 4 slots per Philox call ------------------------------------------
        constexpr int NQ = TILE / (4 * PIC1D_NT);  // quads per thread
        const bool tile_full = tbase + TILE <= n_sorted;  // block-uniform
        unsigned bits = 0;  // bit 4 q + c: slot c of the thread's quad q is a candidate
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            // a thread owns 4 NQ CONSECUTIVE slots, so the candidate list below comes out in slot order and
            // the per-candidate phase reads neighbouring velocities
            const int rel0 = (tid * NQ + q) * 4, i0 = tbase + rel0;
            if (tile_full || i0 < n_sorted) {
                float4 A, B, C;
                if (STAGE) {  // buffers have capacity slots (a multiple of 4096): the vector never leaves them
                    A = *reinterpret_cast<const float4*>(a.vx + i0);
                    B = *reinterpret_cast<const float4*>(a.vy + i0);
                    C = *reinterpret_cast<const float4*>(a.vz + i0);
                }
                uint32_t w[4];
                philox4x32_10((uint32_t)(i0 >> 2), a.step, str_null, 0u, a.k0, a.k1, w);
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    if ((tile_full || i0 + c < n_sorted) && w[c] <= a.null_le) bits |= 1u << (4 * q + c);
                if (a.mask) *reinterpret_cast<uchar4*>(a.mask + i0) = make_uchar4(0, 0, 0, 0);  // 4-aligned, capacity slots
                if (STAGE) {
                    *reinterpret_cast<float4*>(s_vx + rel0) = A;
                    *reinterpret_cast<float4*>(s_vy + rel0) = B;
                    *reinterpret_cast<float4*>(s_vz + rel0) = C;
                }
            }
        }
        if (!a.null_any) bits = 0;
        {
            // append the thread's candidates to the shared list (any order: each is handled on its own)
            const int cnt = __popc(bits);
            int inc = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            int base = 0;
            if (lane == 31 && inc) base = atom_shared_add(&s_n[0], inc);
            base = __shfl_sync(0xffffffffu, base, 31) + inc - cnt;
            if (STAGE) {  // most slots are candidates: predicated stores
#pragma unroll
                for (int b = 0; b < 4 * NQ; ++b)
                    if ((bits >> b) & 1u) s_cand[base++] = (unsigned short)(tid * (4 * NQ) + b);
            } else {      // few are: walk the set bits
                while (bits) {
                    const int b = __ffs(bits) - 1;
                    bits &= bits - 1;
                    s_cand[base++] = (unsigned short)(tid * (4 * NQ) + b);
                }
            }
        }
        __syncthreads();
        // ---- phase B: process selection, one thread per candidate ----------------------------------
        const int n_cand = s_n[0];
        c_cand += (tid < n_cand % PIC1D_NT ? 1 : 0) + n_cand / PIC1D_NT;
        unsigned c_pack = 0;  // four 8-bit event counters of this tile (<= 16 candidates per thread)
        for (int j0 = 0; j0 < n_cand; j0 += PIC1D_NT) {
            const int j = j0 + tid;
            int e = 0;
            int rel = 0;
            if (j < n_cand) {
                rel = s_cand[j];
                const int i = tbase + rel;
                const float vx = STAGE ? s_vx[rel] : a.vx[i], vy = STAGE ? s_vy[rel] : a.vy[i], vz = STAGE ? s_vz[rel] : a.vz[i];
                uint32_t b0[4];
                philox4x32_10((uint32_t)i, a.step, str_coll, 0u, a.k0, a.k1, b0);
                const float u_type = u01(b0[0]);
                const float g2 = __fadd_rn(__fadd_rn(__fmul_rn(vx, vx), __fmul_rn(vy, vy)), __fmul_rn(vz, vz));
                const float g = sqrtf(g2);
                const float aa = __fmul_rn(g, a.inv_g_cap);
                if (aa > 1.0f) ++c_over;
                if (KIND == 1) {
                    // cumulative selection, evaluated lazily: the same operations as the full form,
                    // only skipped where their result cannot matter (P_exc = P_ion = 0 below E_exc)
                    const float En = __fmul_rn(a.c_eV, g2);
                    const float t1 = __fmul_rn(aa, a.r_el);
                    if (u_type < t1) {
                        e = 1;
                    } else if (En > a.E_exc) {
                        const float P_exc = __fmul_rn(__fmul_rn(aa, a.r_exc), __fsub_rn(1.0f, __fdiv_rn(a.E_exc, En)));
                        const float t2 = __fadd_rn(t1, P_exc);
                        if (u_type < t2) {
                            e = 2;
                        } else {
                            const float P_ion = En > a.E_ion
                                ? __fmul_rn(__fmul_rn(aa, a.r_ion), __fsub_rn(1.0f, __fdiv_rn(a.E_ion, En))) : 0.0f;
                            e = u_type < __fadd_rn(t2, P_ion) ? 3 : 0;
                        }
                    }
                } else {  // ion charge exchange with the cold background gas
                    e = u_type < fminf(1.0f, aa) ? 1 : 0;
                }
                c_pack += 1u << (8 * e);
                if (e == 3) atomicOr(&s_ionbits[rel >> 5], 1u << (rel & 31));
                if (a.mask && e) a.mask[i] = (uint8_t)e;
            }
            const int idx = warp_append(e != 0, &s_n[1]);
            if (e) s_coll[idx] = (unsigned short)(rel | (e << 12));
            if (KIND == 1 && __any_sync(0xffffffffu, e == 3)) warp_append(e == 3, &s_n[2]);
        }
        c_e0 += c_pack & 0xff; c_e1 += (c_pack >> 8) & 0xff; c_e2 += (c_pack >> 16) & 0xff; c_e3 += c_pack >> 24;
        __syncthreads();
        // ---- ionisations of the tile: count now, records in phase C, the pairs themselves in k_mcc_births
        const int nb = s_n[2];
        if (KIND == 1 && tid == 0) a.rec_nb[tile] = nb;
        // ---- phase C: kinematics, one thread per real collision -------------------------------------
        const int n_coll = s_n[1];
        for (int j = tid; j < n_coll; j += PIC1D_NT) {
            const int rel = s_coll[j] & 0xfff, e = s_coll[j] >> 12;
            const int i = tbase + rel;
            uint32_t b0[4];
            philox4x32_10((uint32_t)i, a.step, str_coll, 0u, a.k0, a.k1, b0);
            const float u_a = u01(b0[1]), u_b = u01(b0[2]), u_c = u01(b0[3]);
            if (KIND == 1) {
                const float vx = STAGE ? s_vx[rel] : a.vx[i], vy = STAGE ? s_vy[rel] : a.vy[i], vz = STAGE ? s_vz[rel] : a.vz[i];
                const float g2 = __fadd_rn(__fadd_rn(__fmul_rn(vx, vx), __fmul_rn(vy, vy)), __fmul_rn(vz, vz));
                const float En = __fmul_rn(a.c_eV, g2);
                float n[3];
                iso_dir(u_a, u_b, n);
                float gp;
                if (e == 1) {
                    const float g = sqrtf(g2);
                    const float dot = __fadd_rn(__fadd_rn(__fmul_rn(n[0], vx), __fmul_rn(n[1], vy)), __fmul_rn(n[2], vz));
                    const float cchi = __fdiv_rn(dot, g);
                    gp = __fmul_rn(g, sqrtf(__fsub_rn(1.0f, __fmul_rn(a.two_mr, __fsub_rn(1.0f, cchi)))));
                } else if (e == 2) {
                    gp = sqrtf(__fdiv_rn(__fsub_rn(En, a.E_exc), a.c_eV));
                } else {
                    gp = sqrtf(__fdiv_rn(__fmul_rn(__fsub_rn(En, a.E_ion), 0.5f), a.c_eV));
                    // rank among the tile's ionisations in slot order
                    int r = __popc(s_ionbits[rel >> 5] & ((1u << (rel & 31)) - 1u));
                    for (int q = 0; q < (rel >> 5); ++q) r += __popc(s_ionbits[q]);
                    a.rec_rel[tbase + r] = rel;
                    a.rec_gp[tbase + r] = gp;
                }
                a.vx[i] = __fmul_rn(gp, n[0]); a.vy[i] = __fmul_rn(gp, n[1]); a.vz[i] = __fmul_rn(gp, n[2]);
            } else {
                uint32_t b1[4];
                philox4x32_10((uint32_t)i, a.step, str_coll, 1u, a.k0, a.k1, b1);
                const float r12 = bm_r(u_a), ph12 = __fmul_rn(6.2831855f, u_b);
                const float r3 = bm_r(u_c), ph3 = __fmul_rn(6.2831855f, u01(b1[0]));
                a.vx[i] = __fmul_rn(a.gvt, __fmul_rn(r12, cosf(ph12)));
                a.vy[i] = __fmul_rn(a.gvt, __fmul_rn(r12, sinf(ph12)));
                a.vz[i] = __fmul_rn(a.gvt, __fmul_rn(r3, cosf(ph3)));
            }
        }
        __syncthreads();
    }
    // event counters: warp reduce, one global add per warp
    {
        int vals[6] = {c_cand, c_e0, c_e1, c_e2, c_e3, c_over};
#pragma unroll
        for (int q = 0; q < 6; ++q) vals[q] = __reduce_add_sync(0xffffffffu, vals[q]);
        if (lane == 0) {
            if (vals[0]) atomicAdd(&sp.n_candidates, (ull)vals[0]);
#pragma unroll
            for (int q = 0; q < 4; ++q) if (vals[1 + q]) atomicAdd(&sp.n_events[q], (ull)vals[1 + q]);
            if (vals[5]) atomicAdd(&sp.over_cap, (ull)vals[5]);
        }
    }
}

// ---- the ionisation pairs (L203), in ascending parent-slot order ---------------------------------------
// k_mcc left, per tile, the number of ionisations and their (parent slot, electron speed) records in slot
// order.  Birth index = (ionisations of all earlier tiles) + (rank inside the tile): every block takes a
// contiguous chunk of tiles, sums the counts of the tiles before its chunk itself (a few 10^4 integers
// from L2, read coalesced) and scans its own chunk -- nobody waits for anybody.  A decoupled look-back
// inside k_mcc did the same job first; it cost 15-20 % of that kernel, because the tiles in flight wait
// for each other's counts at a barrier (profiles/r1_notes.md).
__global__ void __launch_bounds__(PIC1D_NT) k_mcc_births(MccArgs a) {
    __shared__ int s_w[PIC1D_NWARP + 1];
    __shared__ int s_pre[PIC1D_NT], s_cnt[PIC1D_NT];
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    DevState* st = a.st;
    const int n_sorted = st->sp[a.s].n_sorted;
    const int n_act = (n_sorted + MCC_TILE - 1) / MCC_TILE;
    const int chunk = (n_act + gridDim.x - 1) / gridDim.x;
    const int t0 = min(blockIdx.x * chunk, n_act), t1 = min(t0 + chunk, n_act);
    if (t0 >= t1) return;
    auto block_sum = [&](int v) -> int {
        v = __reduce_add_sync(0xffffffffu, v);
        __syncthreads();
        if (lane == 0) s_w[wp] = v;
        __syncthreads();
        int t = 0;
#pragma unroll
        for (int q = 0; q < PIC1D_NWARP; ++q) t += s_w[q];
        return t;
    };
    int part = 0;
    for (int t = tid; t < t0; t += PIC1D_NT) part += a.rec_nb[t];
    int base = block_sum(part);  // ionisations of the tiles before this block's chunk
    const int ne = st->sp[0].n_sorted, ni = a.n_species > 1 ? st->sp[1].n_sorted : 0;
    int room = a.cap_e - ne;
    if (a.n_species > 1) room = min(room, a.cap_i - ni);
    const uint32_t str_coll = STREAM_COLL + (uint32_t)a.s;
    for (int c0 = t0; c0 < t1; c0 += PIC1D_NT) {
        const int nt = min(PIC1D_NT, t1 - c0);
        const int v = tid < nt ? a.rec_nb[c0 + tid] : 0;
        int inc = v;  // exclusive scan of the piece's counts
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        __syncthreads();
        if (lane == 31) s_w[wp] = inc;
        __syncthreads();
        int before = 0, tot = 0;
#pragma unroll
        for (int q = 0; q < PIC1D_NWARP; ++q) { const int u = s_w[q]; if (q < wp) before += u; tot += u; }
        s_pre[tid] = base + before + inc - v;
        s_cnt[tid] = v;
        __syncthreads();
        for (int q = wp; q < nt; q += PIC1D_NWARP) {  // one warp per tile
            const int nbq = s_cnt[q], tbase = (c0 + q) * MCC_TILE;
            for (int r = lane; r < nbq; r += 32) {
                const int b = s_pre[q] + r;  // birth index of the step, ascending parent slot
                if (b >= room) continue;
                const uint32_t i = (uint32_t)(tbase + a.rec_rel[tbase + r]);
                uint32_t b0[4], b1[4], b2[4];
                philox4x32_10(i, a.step, str_coll, 0u, a.k0, a.k1, b0);
                philox4x32_10(i, a.step, str_coll, 1u, a.k0, a.k1, b1);
                philox4x32_10(i, a.step, str_coll, 2u, a.k0, a.k1, b2);
                const float xp = a.x[i];
                float n2[3];
                iso_dir(u01(b0[3]), u01(b1[0]), n2);
                const float gp = a.rec_gp[tbase + r];
                const int de = ne + b;
                a.ex[de] = xp;
                a.evx[de] = __fmul_rn(gp, n2[0]); a.evy[de] = __fmul_rn(gp, n2[1]); a.evz[de] = __fmul_rn(gp, n2[2]);
                if (a.n_species > 1) {
                    const float r12 = bm_r(u01(b1[1])), ph12 = __fmul_rn(6.2831855f, u01(b1[2]));
                    const float r3 = bm_r(u01(b1[3])), ph3 = __fmul_rn(6.2831855f, u01(b2[0]));
                    const int di = ni + b;
                    a.ix[di] = xp;
                    a.ivx[di] = __fmul_rn(a.gvt, __fmul_rn(r12, cosf(ph12)));
                    a.ivy[di] = __fmul_rn(a.gvt, __fmul_rn(r12, sinf(ph12)));
                    a.ivz[di] = __fmul_rn(a.gvt, __fmul_rn(r3, cosf(ph3)));
                }
            }
        }
        base += tot;
        __syncthreads();
    }
    if (t1 == n_act && tid == 0) {  // the block with the last tile closes the step's birth bookkeeping
        const int total = base;
        const int kept = min(total, max(room, 0));
        st->sp[0].n_live = ne + kept;
        st->sp[0].births += (ull)kept;
        if (a.n_species > 1) {
            st->sp[1].n_live = ni + kept;
            st->sp[1].births += (ull)kept;
        }
        if (total > kept) {
            st->sp[0].dropped += (ull)(total - kept);
            if (a.n_species > 1) st->sp[1].dropped += (ull)(total - kept);
            atomicOr(&st->err, ERRBIT_CAPACITY);
        }
    }
}
