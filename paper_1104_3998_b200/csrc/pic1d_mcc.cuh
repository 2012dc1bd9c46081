// pic1d_mcc.cuh -- modified null-collision Monte-Carlo collisions (Eq. 6).
//
// Every sorted particle draws p (L203); p < P0 enters the standard null-collision selection with the
// synthetic analytic cross sections (products and sums only, in the spirit of L207).  The particle id
// is the slot in the sorted array (R18), so the collisions can run wherever that slot is known:
//
//   folded             mcc_lane(): inside the scatter kernels of the fine sort, where the destination
//                      slot of a particle IS its id and vx, vy, vz are still in registers / shared memory
//                      (the paper fuses for the same reason, L182: "re-use particle
//                      data ... reduce the memory transfer").  MCC reads neither rho nor E, so running it
//                      before the deposit and the field solve changes nothing (R3).
//   stand-alone        k_mcc: a pass over the sorted arrays after the field solve.  The paper notes that
//                      this module has "lots of branches" (L209); here the branches are removed by
//                      compaction inside a tile of MCC_TILE sorted slots:
//                        phase A  null test for every slot: one Philox call serves 4 consecutive slots
//                                 (R12); nothing is loaded; candidates -> shared list
//                        phase B  one thread per CANDIDATE: load v, Philox, process selection
//                        phase C  one thread per REAL COLLISION: kinematics, velocity written back
//   k_mcc_births       one thread per IONISATION: the new electron / ion pair (both variants).
//
// Ionisation products go to the tails of the electron / ion arrays in ascending parent-slot order (the
// paper allocates them with a shared counter inside the parent's sort cell, L203; here the tail is sorted
// into place by the next step's fine sort).  Whoever finds an ionisation sets the parent's bit in a bit
// mask over the sorted slots, stores the pair's electron speed at the parent's slot and counts it per
// tile of MCC_TILE slots; k_mcc_births orders the births by walking the bit mask -- no atomic decides an
// index (the per-tile counter is a sum, its order carries no meaning).
#pragma once
#include "pic1d_device.cuh"

#define MCC_TILE (PIC1D_NT * 16)  // sorted slots per tile

// Parameters of the collision model, shared by k_mcc and by the scatter kernels that fold it in.
struct MccP {
    DevState* st;
    uint8_t* mask;       // optional event mask per sorted slot (PIC1D_FLAG_CAPTURE)
    unsigned* ion_bits;  // electron set: bit per sorted slot "ionised in this step"; all zero between steps
    float* ion_gp;       // electron set: [slot] speed shared by the two electrons of the slot's ionisation
    int* ion_nb;         // electron set: [slot / MCC_TILE] ionisations of the tile; zeroed by k_step_begin
    unsigned* null_bits; // folded variant: bit per sorted slot "passes the null test in this step" (k_null_bits)
    int s, kind;
    uint32_t k0, k1;
    uint32_t null_le;    // null test in integers: U(w) < P0  <=>  w <= null_le   (null_any = 0: never)
    int null_any;
    float inv_g_cap, c_eV, r_el, r_exc, r_ion, E_exc, E_ion, two_mr, gvt;
};

struct MccArgs {
    float *x, *vx, *vy, *vz;      // this species' current (sorted) buffer
    float *ex, *evx, *evy, *evz;  // electron buffer (birth tail)
    float *ix, *ivx, *ivy, *ivz;  // ion buffer (birth tail), may be null
    MccP m;
    int n_species, cap_e, cap_i;
};

// per-thread event counters, packed (a thread sees < 65536 particles per launch)
struct MccCount {
    unsigned cand_e1;  // candidates | elastic or CX << 16
    unsigned e2_e3;    // excitations | ionisations << 16
    unsigned over;     // candidates with g > g_cap
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

// Process selection of one candidate (R13): mul / add / div / sqrt / compare only, so the event
// is bit-exact.  Evaluated lazily: the same operations as the full cumulative form, skipped only where
// their result cannot matter (P_exc = P_ion = 0 below E_exc).  Returns 0 null, 1 elastic / CX,
// 2 excitation, 3 ionisation; over = candidate with g > g_cap.
template <int KIND>
__device__ __forceinline__ int mcc_select(const MccP& m, float vx, float vy, float vz, float u_type, bool& over) {
    const float g2 = __fadd_rn(__fadd_rn(__fmul_rn(vx, vx), __fmul_rn(vy, vy)), __fmul_rn(vz, vz));
    const float g = sqrtf(g2);
    const float aa = __fmul_rn(g, m.inv_g_cap);
    over = aa > 1.0f;
    if (KIND == 1) {
        const float En = __fmul_rn(m.c_eV, g2);
        const float t1 = __fmul_rn(aa, m.r_el);
        if (u_type < t1) return 1;
        if (!(En > m.E_exc)) return 0;
        const float P_exc = __fmul_rn(__fmul_rn(aa, m.r_exc), __fsub_rn(1.0f, __fdiv_rn(m.E_exc, En)));
        const float t2 = __fadd_rn(t1, P_exc);
        if (u_type < t2) return 2;
        const float P_ion = En > m.E_ion
            ? __fmul_rn(__fmul_rn(aa, m.r_ion), __fsub_rn(1.0f, __fdiv_rn(m.E_ion, En))) : 0.0f;
        return u_type < __fadd_rn(t2, P_ion) ? 3 : 0;
    }
    return u_type < fminf(1.0f, aa) ? 1 : 0;  // ion charge exchange with the cold background gas
}

// Post-collision velocity of an electron event e in {1, 2, 3} (R14); returns the new speed.
__device__ __forceinline__ float mcc_electron_kinematics(const MccP& m, int e, float& vx, float& vy, float& vz,
                                                         float u_a, float u_b) {
    const float g2 = __fadd_rn(__fadd_rn(__fmul_rn(vx, vx), __fmul_rn(vy, vy)), __fmul_rn(vz, vz));
    const float En = __fmul_rn(m.c_eV, g2);
    float n[3];
    iso_dir(u_a, u_b, n);
    float gp;
    if (e == 1) {
        const float g = sqrtf(g2);
        const float dot = __fadd_rn(__fadd_rn(__fmul_rn(n[0], vx), __fmul_rn(n[1], vy)), __fmul_rn(n[2], vz));
        const float cchi = __fdiv_rn(dot, g);
        gp = __fmul_rn(g, sqrtf(__fsub_rn(1.0f, __fmul_rn(m.two_mr, __fsub_rn(1.0f, cchi)))));
    } else if (e == 2) {
        gp = sqrtf(__fdiv_rn(__fsub_rn(En, m.E_exc), m.c_eV));
    } else {
        gp = sqrtf(__fdiv_rn(__fmul_rn(__fsub_rn(En, m.E_ion), 0.5f), m.c_eV));
    }
    vx = __fmul_rn(gp, n[0]); vy = __fmul_rn(gp, n[1]); vz = __fmul_rn(gp, n[2]);
    return gp;
}

// Maxwellian gas velocity gvt N(0,1)^3 from four uniforms (Box-Muller; charge exchange and new ions)
__device__ __forceinline__ void mcc_gas_velocity(float gvt, float u1, float u2, float u3, float u4,
                                                 float& vx, float& vy, float& vz) {
    const float r12 = bm_r(u1), ph12 = __fmul_rn(6.2831855f, u2);
    const float r3 = bm_r(u3), ph3 = __fmul_rn(6.2831855f, u4);
    vx = __fmul_rn(gvt, __fmul_rn(r12, cosf(ph12)));
    vy = __fmul_rn(gvt, __fmul_rn(r12, sinf(ph12)));
    vz = __fmul_rn(gvt, __fmul_rn(r3, cosf(ph3)));
}

// an ionisation of sorted slot i: bit, pair speed, per-tile count (k_mcc_births orders the births)
__device__ __forceinline__ void mcc_record_ionisation(const MccP& m, unsigned i, float gp) {
    atomicOr(&m.ion_bits[i >> 5], 1u << (i & 31u));
    m.ion_gp[i] = gp;
    atomicAdd(&m.ion_nb[i / MCC_TILE], 1);
}

// ---- folded variant: pieces the scatter kernels call -------------------------------------------------
// The null test of slot d depends on (seed, step, species, d) only, so it is evaluated ahead of the scatter
// for ALL slots by k_null_bits -- one Philox call per 4 consecutive slots, exactly the draw of DESIGN.md R12
// -- and the scatter looks its destination slot up in the bit mask (L2-resident: capacity / 8 bytes).
__device__ __forceinline__ bool mcc_null_bit(const MccP& m, unsigned d) {
    return (__ldcg(m.null_bits + (d >> 5)) >> (d & 31u)) & 1u;
}

// process selection of the candidate in slot d (cand = false: the lane idles through the same code);
// counts the event; returns it.  Same draws as k_mcc: philox(d, step, COLL + s, 0).
template <int KIND>
__device__ __forceinline__ int mcc_event(const MccP& m, uint32_t step, unsigned d, bool cand,
                                         float vx, float vy, float vz, MccCount& c, uint32_t (&b0)[4]) {
    philox4x32_10(d, step, STREAM_COLL + (uint32_t)m.s, 0u, m.k0, m.k1, b0);
    int e = 0;
    if (cand) {
        bool over;
        e = mcc_select<KIND>(m, vx, vy, vz, u01(b0[0]), over);
        c.cand_e1 += 1u + (e == 1 ? 0x10000u : 0u);
        c.e2_e3 += (e == 2 ? 1u : 0u) + (e == 3 ? 0x10000u : 0u);
        c.over += over ? 1u : 0u;
    }
    return e;
}

// kinematics of the real collision e != 0 in slot d, given the words b0 of philox(d, step, COLL + s, 0)
template <int KIND>
__device__ __forceinline__ void mcc_kinematics(const MccP& m, uint32_t step, unsigned d, int e, const uint32_t (&b0)[4],
                                               float& vx, float& vy, float& vz) {
    if (KIND == 1) {
        const float gp = mcc_electron_kinematics(m, e, vx, vy, vz, u01(b0[1]), u01(b0[2]));
        if (e == 3) mcc_record_ionisation(m, d, gp);
    } else {
        uint32_t b1[4];
        philox4x32_10(d, step, STREAM_COLL + (uint32_t)m.s, 1u, m.k0, m.k1, b1);
        mcc_gas_velocity(m.gvt, u01(b0[1]), u01(b0[2]), u01(b0[3]), u01(b1[0]), vx, vy, vz);
    }
}

// The collisions of ONE particle whose sorted slot d is known, start to finish.  Must be called by all 32
// lanes (cand = the lane holds a particle that goes to slot d and passed the null test).
template <int KIND>
__device__ __forceinline__ int mcc_lane(const MccP& m, uint32_t step, unsigned d, bool cand,
                                        float& vx, float& vy, float& vz, MccCount& c) {
    int e = 0;
    if (__any_sync(0xffffffffu, cand)) {
        uint32_t b0[4];
        e = mcc_event<KIND>(m, step, d, cand, vx, vy, vz, c, b0);
        if (e) mcc_kinematics<KIND>(m, step, d, e, b0, vx, vy, vz);
    }
    return e;
}

// null-test bit mask of the species for this step: bit d = slot d is a candidate.  One thread per word of
// 32 slots (8 Philox calls); called from the extra blocks of k_bin_scan, between count and scatter.
__device__ __forceinline__ void mcc_null_words(const MccP& m, int wd) {
    const int n_src = m.st->sp[m.s].n_src;  // the sorted part will not be longer than the source
    if (wd >= ((n_src + 31) >> 5)) return;
    const uint32_t step = m.st->step;
    unsigned bits = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        uint32_t w[4];
        philox4x32_10((uint32_t)(wd * 8 + q), step, STREAM_NULL + (uint32_t)m.s, 0u, m.k0, m.k1, w);
#pragma unroll
        for (int c = 0; c < 4; ++c) bits |= (w[c] <= m.null_le ? 1u : 0u) << (4 * q + c);
    }
    m.null_bits[wd] = m.null_any ? bits : 0u;
}

// The same mask one step AHEAD: the null test of slot d depends on (seed, step, species, d) only, so the mask of step
// n + 1 is computed while step n's electron sort runs (side stream; that kernel leaves most issue slots idle) and
// the extra blocks of k_bin_scan are not needed.  It runs after the births, so the species' n_live is the next step's
// source count -- except for electrons, which may still receive secondaries: all capacity / 32 words for them.
__global__ void __launch_bounds__(256) k_null_bits_next(MccP m, int n_words) {
    const int wd = blockIdx.x * blockDim.x + threadIdx.x;
    if (m.s != 0) n_words = min(n_words, (m.st->sp[m.s].n_live + 31) >> 5);
    if (wd >= n_words) return;
    const uint32_t step = m.st->step_next;
    unsigned bits = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        uint32_t w[4];
        philox4x32_10((uint32_t)(wd * 8 + q), step, STREAM_NULL + (uint32_t)m.s, 0u, m.k0, m.k1, w);
#pragma unroll
        for (int c = 0; c < 4; ++c) bits |= (w[c] <= m.null_le ? 1u : 0u) << (4 * q + c);
    }
    m.null_bits[wd] = m.null_any ? bits : 0u;
}

// warp-reduce the packed per-thread counters and add them to the species' cumulative counters
__device__ __forceinline__ void mcc_flush_counts(const MccP& m, const MccCount& c) {
    int vals[5] = {(int)(c.cand_e1 & 0xffffu), (int)(c.cand_e1 >> 16), (int)(c.e2_e3 & 0xffffu), (int)(c.e2_e3 >> 16), (int)c.over};
#pragma unroll
    for (int q = 0; q < 5; ++q) vals[q] = __reduce_add_sync(0xffffffffu, vals[q]);
    if ((threadIdx.x & 31) == 0 && (vals[0] | vals[1] | vals[2] | vals[3] | vals[4])) {
        DevSpecies& sp = m.st->sp[m.s];
        if (vals[0]) atomicAdd(&sp.n_candidates, (ull)vals[0]);
        const int nulls = vals[0] - vals[1] - vals[2] - vals[3];  // may be negative when the candidates are added elsewhere
        if (nulls) atomicAdd(&sp.n_events[0], (ull)(long long)nulls);
#pragma unroll
        for (int q = 1; q < 4; ++q) if (vals[q]) atomicAdd(&sp.n_events[q], (ull)vals[q]);
        if (vals[4]) atomicAdd(&sp.over_cap, (ull)vals[4]);
    }
}

// append `flag`-ged items of a warp to a shared list; returns this lane's index (valid if flag)
__device__ __forceinline__ int warp_append(bool flag, int* counter) {
    const unsigned bal = __ballot_sync(0xffffffffu, flag);
    int base = 0;
    if ((threadIdx.x & 31) == 0 && bal) base = atom_shared_add(counter, __popc(bal));
    base = __shfl_sync(0xffffffffu, base, 0);
    return base + __popc(bal & lanemask_lt());
}

// ---- bulk asynchronous copies (TMA engine, non-tensor form) + mbarrier ------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// ---- stand-alone pass over the sorted arrays -----------------------------------------------------------
// KIND: 1 electron set, 2 ion charge exchange.  Persistent blocks take tiles of MCC_TILE sorted slots by
// ticket.  STAGE (species most of whose particles are candidates): the tile's vx, vy, vz are streamed into
// shared memory by three bulk asynchronous copies (cp.async.bulk, completion on an mbarrier) that fly while
// phase A computes the null tests, so phases B / C never wait for a gathered global load; otherwise phases
// B / C fetch the few candidates' velocities from global memory.
template <int KIND, bool STAGE>
__global__ void __launch_bounds__(PIC1D_NT, STAGE ? 3 : 4) k_mcc(MccArgs a) {
    constexpr int TILE = MCC_TILE;
    extern __shared__ __align__(128) float s_v[];  // STAGE: [3][TILE]
    __shared__ unsigned long long s_bar;
    __shared__ int s_tile;
    __shared__ int s_n[2];                   // candidates, real collisions
    __shared__ unsigned short s_cand[TILE];  // slot - tile base
    __shared__ unsigned short s_coll[TILE];  // (slot - tile base) | event << 12
    const int tid = threadIdx.x, lane = tid & 31;
    const MccP& m = a.m;
    DevState* st = m.st;
    DevSpecies& sp = st->sp[m.s];
    const int n_sorted = sp.n_sorted;
    const int n_act = (n_sorted + TILE - 1) / TILE;
    const uint32_t step = st->step;
    const uint32_t str_null = STREAM_NULL + (uint32_t)m.s, str_coll = STREAM_COLL + (uint32_t)m.s;
    MccCount cnt = {0u, 0u, 0u};
    ull n_cand_block = 0;  // thread 0: candidates of the block's tiles (the list lengths)
    unsigned parity = 0;
    if (STAGE && tid == 0) mbar_init(&s_bar, 1);
    while (true) {
        if (tid == 0) {
            const int t = atomicAdd(&sp.ticket, 1);
            s_tile = t; s_n[0] = 0; s_n[1] = 0;
            if (STAGE && t < n_act) {  // the arrays hold capacity slots, a multiple of TILE: a whole tile is always in bounds
                mbar_expect_tx(&s_bar, 3u * TILE * sizeof(float));
                bulk_g2s(s_v, a.vx + (size_t)t * TILE, TILE * sizeof(float), &s_bar);
                bulk_g2s(s_v + TILE, a.vy + (size_t)t * TILE, TILE * sizeof(float), &s_bar);
                bulk_g2s(s_v + 2 * TILE, a.vz + (size_t)t * TILE, TILE * sizeof(float), &s_bar);
            }
        }
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
                uint32_t w[4];
                philox4x32_10((uint32_t)(i0 >> 2), step, str_null, 0u, m.k0, m.k1, w);
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    if ((tile_full || i0 + c < n_sorted) && w[c] <= m.null_le) bits |= 1u << (4 * q + c);
                if (m.mask) *reinterpret_cast<uchar4*>(m.mask + i0) = make_uchar4(0, 0, 0, 0);  // 4-aligned, capacity slots
            }
        }
        if (!m.null_any) bits = 0;
        {
            // append the thread's candidates to the shared list (any order: each is handled on its own)
            const int cn = __popc(bits);
            int inc = cn;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            int base = 0;
            if (lane == 31 && inc) base = atom_shared_add(&s_n[0], inc);
            base = __shfl_sync(0xffffffffu, base, 31) + inc - cn;
            while (bits) {  // walk the set bits
                const int b = __ffs(bits) - 1;
                bits &= bits - 1;
                s_cand[base++] = (unsigned short)(tid * (4 * NQ) + b);
            }
        }
        __syncthreads();
        if (STAGE) { mbar_wait(&s_bar, parity); parity ^= 1u; }
        // ---- phase B: process selection, one thread per candidate ----------------------------------
        const int n_cand = s_n[0];
        for (int j0 = 0; j0 < n_cand; j0 += PIC1D_NT) {
            const int j = j0 + tid;
            int e = 0;
            int rel = 0;
            if (j < n_cand) {
                rel = s_cand[j];
                const int i = tbase + rel;
                const float vx = STAGE ? s_v[rel] : a.vx[i], vy = STAGE ? s_v[TILE + rel] : a.vy[i],
                            vz = STAGE ? s_v[2 * TILE + rel] : a.vz[i];
                uint32_t b0[4];
                philox4x32_10((uint32_t)i, step, str_coll, 0u, m.k0, m.k1, b0);
                bool over;
                e = mcc_select<KIND>(m, vx, vy, vz, u01(b0[0]), over);
                cnt.over += over ? 1u : 0u;  // (the events are counted by phase C, the candidates per tile)
            }
            const int idx = warp_append(e != 0, &s_n[1]);
            if (e) s_coll[idx] = (unsigned short)(rel | (e << 12));
        }
        __syncthreads();
        // ---- phase C: kinematics, one thread per real collision -------------------------------------
        const int n_coll = s_n[1];
        if (tid == 0) n_cand_block += (ull)n_cand;
        for (int j = tid; j < n_coll; j += PIC1D_NT) {
            const int rel = s_coll[j] & 0xfff, e = s_coll[j] >> 12;
            const int i = tbase + rel;
            cnt.cand_e1 += e == 1 ? 0x10000u : 0u;
            cnt.e2_e3 += (e == 2 ? 1u : 0u) + (e == 3 ? 0x10000u : 0u);
            if (m.mask) m.mask[i] = (uint8_t)e;
            uint32_t b0[4];
            philox4x32_10((uint32_t)i, step, str_coll, 0u, m.k0, m.k1, b0);
            float vx, vy, vz;
            if (KIND == 1) {
                vx = STAGE ? s_v[rel] : a.vx[i]; vy = STAGE ? s_v[TILE + rel] : a.vy[i]; vz = STAGE ? s_v[2 * TILE + rel] : a.vz[i];
                const float gp = mcc_electron_kinematics(m, e, vx, vy, vz, u01(b0[1]), u01(b0[2]));
                if (e == 3) mcc_record_ionisation(m, (unsigned)i, gp);
            } else {
                uint32_t b1[4];
                philox4x32_10((uint32_t)i, step, str_coll, 1u, m.k0, m.k1, b1);
                mcc_gas_velocity(m.gvt, u01(b0[1]), u01(b0[2]), u01(b0[3]), u01(b1[0]), vx, vy, vz);
            }
            a.vx[i] = vx; a.vy[i] = vy; a.vz[i] = vz;
        }
        __syncthreads();
    }
    mcc_flush_counts(m, cnt);  // events and over-cap; its null count is (0 candidates - events) ...
    if (tid == 0 && n_cand_block) {  // ... and the candidates complete both (unsigned wrap-around is exact)
        atomicAdd(&sp.n_candidates, n_cand_block);
        atomicAdd(&sp.n_events[0], n_cand_block);
    }
}

// ---- the ionisation pairs (L203), in ascending parent-slot order ---------------------------------------
// The collisions left a bit per ionising sorted slot, the pair's electron speed at that slot, and the
// number of ionisations per tile of MCC_TILE slots.  Birth index = (ionisations of all earlier tiles) +
// (rank inside the tile): every block takes a contiguous chunk of tiles, sums the counts of the tiles
// before its chunk itself (a few 10^4 integers from L2, read coalesced) and scans its own chunk -- nobody
// waits for anybody.  Inside a tile one warp walks the bit mask in quarters of 1024 slots (one word per
// lane): prefix of the popcounts, the set bits go to a shared list in slot order, then one lane per birth.
// The bits are cleared on the way (they are all zero between steps).
// A decoupled look-back inside k_mcc did this job first; it cost 15-20 % of that kernel, because the tiles
// in flight wait for each other's counts at a barrier (profiles/r1_notes.md).
__global__ void __launch_bounds__(PIC1D_NT) k_mcc_births(MccArgs a) {
    __shared__ int s_w[PIC1D_NWARP + 1];
    __shared__ int s_pre[PIC1D_NT], s_cnt[PIC1D_NT];
    __shared__ unsigned short s_list[PIC1D_NWARP][1024];
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    const MccP& m = a.m;
    DevState* st = m.st;
    const int n_sorted = st->sp[m.s].n_sorted;
    const int n_act = (n_sorted + MCC_TILE - 1) / MCC_TILE;
    const int chunk = (n_act + gridDim.x - 1) / gridDim.x;
    const int t0 = min(blockIdx.x * chunk, n_act), t1 = min(t0 + chunk, n_act);
    const int ne = st->sp[0].n_sorted, ni = a.n_species > 1 ? st->sp[1].n_sorted : 0;
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
    for (int t = tid; t < t0; t += PIC1D_NT) part += m.ion_nb[t];
    int base = block_sum(part);  // ionisations of the tiles before this block's chunk
    int room = a.cap_e - ne;
    if (a.n_species > 1) room = min(room, a.cap_i - ni);
    const uint32_t step = st->step;
    const uint32_t str_coll = STREAM_COLL + (uint32_t)m.s;
    for (int c0 = t0; c0 < t1; c0 += PIC1D_NT) {
        const int nt = min(PIC1D_NT, t1 - c0);
        const int v = tid < nt ? m.ion_nb[c0 + tid] : 0;
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
            if (s_cnt[q] == 0) continue;
            const int tbase = (c0 + q) * MCC_TILE;
            int b_tile = s_pre[q];  // birth index of the tile's first ionisation
            for (int quarter = 0; quarter < MCC_TILE / 1024; ++quarter) {
                const int wbase = tbase + quarter * 1024;  // the quarter's first slot
                unsigned* wordp = m.ion_bits + (wbase >> 5) + lane;
                unsigned word = *wordp;
                if (!__any_sync(0xffffffffu, word != 0u)) continue;
                if (word) *wordp = 0u;
                const int pc = __popc(word);
                int pinc = pc;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int t = __shfl_up_sync(0xffffffffu, pinc, o);
                    if (lane >= o) pinc += t;
                }
                const int nq = __shfl_sync(0xffffffffu, pinc, 31);
                int li = pinc - pc;
                while (word) {  // the lane's set bits, ascending
                    const int bpos = __ffs(word) - 1;
                    word &= word - 1;
                    s_list[wp][li++] = (unsigned short)(lane * 32 + bpos);
                }
                __syncwarp();
                for (int r = lane; r < nq; r += 32) {
                    const int b = b_tile + r;  // birth index of the step, ascending parent slot
                    if (b >= room) continue;
                    const uint32_t i = (uint32_t)(wbase + s_list[wp][r]);
                    uint32_t b0[4], b1[4], b2[4];
                    philox4x32_10(i, step, str_coll, 0u, m.k0, m.k1, b0);
                    philox4x32_10(i, step, str_coll, 1u, m.k0, m.k1, b1);
                    philox4x32_10(i, step, str_coll, 2u, m.k0, m.k1, b2);
                    const float xp = a.x[i];
                    float n2[3];
                    iso_dir(u01(b0[3]), u01(b1[0]), n2);
                    const float gp = m.ion_gp[i];
                    const int de = ne + b;
                    a.ex[de] = xp;
                    a.evx[de] = __fmul_rn(gp, n2[0]); a.evy[de] = __fmul_rn(gp, n2[1]); a.evz[de] = __fmul_rn(gp, n2[2]);
                    if (a.n_species > 1) {
                        const int di = ni + b;
                        float wx, wy, wz;
                        mcc_gas_velocity(m.gvt, u01(b1[1]), u01(b1[2]), u01(b1[3]), u01(b2[0]), wx, wy, wz);
                        a.ix[di] = xp; a.ivx[di] = wx; a.ivy[di] = wy; a.ivz[di] = wz;
                    }
                }
                __syncwarp();
                b_tile += nq;
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
