// pic1d_mcc.cuh -- modified null-collision Monte-Carlo collisions (Eq. 6).
//
// Every sorted particle draws p (L203); p < P0 enters the standard null-collision selection with the
// synthetic analytic cross sections (products and sums only, in the spirit of L207).  One thread
// handles 4 consecutive sorted slots, so one Philox call serves their 4 null tests (R12).
// Ionisation products go to the tails of the electron / ion arrays in ascending parent-slot order
// (the paper allocates them with a shared counter inside the parent's sort cell, L203; here the tail
// is sorted into place by the next step's fine sort).  The cross-block order comes from a decoupled
// look-back over per-block ionisation counts -- no atomics decide any index.
#pragma once
#include "pic1d_device.cuh"

#define MCC_TILE (PIC1D_NT * 4)

struct MccArgs {
    float *x, *vx, *vy, *vz;      // this species' current (sorted) buffer
    float *ex, *evx, *evy, *evz;  // electron buffer (birth tail)
    float *ix, *ivx, *ivy, *ivz;  // ion buffer (birth tail), may be null
    DevState* st;
    ull* desc;       // look-back descriptors, one per tile
    uint8_t* mask;   // optional event mask per sorted slot
    int s, kind, n_species, cap_e, cap_i;
    uint32_t step, k0, k1;
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

#define DESC_AGG 1ull
#define DESC_PREFIX 2ull
__device__ __forceinline__ ull desc_pack(uint32_t epoch, ull flag, int v) {
    return ((ull)epoch << 32) | (flag << 30) | (ull)(unsigned)v;
}

__global__ void __launch_bounds__(PIC1D_NT) k_mcc(MccArgs a) {
    __shared__ int s_tile, s_excl;
    __shared__ int s_w[PIC1D_NWARP];
    __shared__ ull s_cnt[6];
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    DevState* st = a.st;
    DevSpecies& sp = st->sp[a.s];
    if (tid == 0) s_tile = atomicAdd(&sp.ticket, 1);
    if (tid < 6) s_cnt[tid] = 0;
    __syncthreads();
    const int tile = s_tile;
    const int n_sorted = sp.n_sorted;
    const int n_act = (n_sorted + MCC_TILE - 1) / MCC_TILE;
    if (tile >= n_act) return;
    const int i0 = tile * MCC_TILE + tid * 4;
    const uint32_t epoch = a.step + 1u;

    int ev[4] = {0, 0, 0, 0};
    float gp_ion[4];
    int n_cand = 0, n_over = 0, n_ion = 0;
    if (i0 < n_sorted) {
        uint32_t w[4];
        philox4x32_10((uint32_t)(i0 >> 2), a.step, STREAM_NULL + (uint32_t)a.s, 0u, a.k0, a.k1, w);
        bool cand[4];
        bool any = false;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            cand[c] = (i0 + c < n_sorted) && (u01(w[c]) < a.P0);
            any |= cand[c];
        }
        if (any) {
            float vx[4], vy[4], vz[4];
            {
                const float4 A = *reinterpret_cast<const float4*>(a.vx + i0);
                const float4 B = *reinterpret_cast<const float4*>(a.vy + i0);
                const float4 C = *reinterpret_cast<const float4*>(a.vz + i0);
                vx[0] = A.x; vx[1] = A.y; vx[2] = A.z; vx[3] = A.w;
                vy[0] = B.x; vy[1] = B.y; vy[2] = B.z; vy[3] = B.w;
                vz[0] = C.x; vz[1] = C.y; vz[2] = C.z; vz[3] = C.w;
            }
            bool changed = false;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                if (!cand[c]) continue;
                ++n_cand;
                const uint32_t i = (uint32_t)(i0 + c);
                uint32_t b0[4];
                philox4x32_10(i, a.step, STREAM_COLL + (uint32_t)a.s, 0u, a.k0, a.k1, b0);
                const float u_type = u01(b0[0]), u_a = u01(b0[1]), u_b = u01(b0[2]), u_c = u01(b0[3]);
                const float g2 = __fadd_rn(__fadd_rn(__fmul_rn(vx[c], vx[c]), __fmul_rn(vy[c], vy[c])),
                                           __fmul_rn(vz[c], vz[c]));
                const float g = sqrtf(g2);
                const float aa = __fmul_rn(g, a.inv_g_cap);
                if (aa > 1.0f) ++n_over;
                if (a.kind == 1) {
                    const float En = __fmul_rn(a.c_eV, g2);
                    const float P_el = __fmul_rn(aa, a.r_el);
                    const float P_exc = En > a.E_exc
                        ? __fmul_rn(__fmul_rn(aa, a.r_exc), __fsub_rn(1.0f, __fdiv_rn(a.E_exc, En))) : 0.0f;
                    const float P_ion = En > a.E_ion
                        ? __fmul_rn(__fmul_rn(aa, a.r_ion), __fsub_rn(1.0f, __fdiv_rn(a.E_ion, En))) : 0.0f;
                    const float t1 = P_el, t2 = __fadd_rn(t1, P_exc), t3 = __fadd_rn(t2, P_ion);
                    const int e = u_type < t1 ? 1 : (u_type < t2 ? 2 : (u_type < t3 ? 3 : 0));
                    ev[c] = e | 4;  // bit 2: was a candidate
                    if (e == 0) continue;
                    float n[3];
                    iso_dir(u_a, u_b, n);
                    float gp;
                    if (e == 1) {
                        const float dot = __fadd_rn(__fadd_rn(__fmul_rn(n[0], vx[c]), __fmul_rn(n[1], vy[c])),
                                                    __fmul_rn(n[2], vz[c]));
                        const float cchi = __fdiv_rn(dot, g);
                        gp = __fmul_rn(g, sqrtf(__fsub_rn(1.0f, __fmul_rn(a.two_mr, __fsub_rn(1.0f, cchi)))));
                    } else if (e == 2) {
                        gp = sqrtf(__fdiv_rn(__fsub_rn(En, a.E_exc), a.c_eV));
                    } else {
                        gp = sqrtf(__fdiv_rn(__fmul_rn(__fsub_rn(En, a.E_ion), 0.5f), a.c_eV));
                        gp_ion[c] = gp;
                        ++n_ion;
                    }
                    vx[c] = __fmul_rn(gp, n[0]); vy[c] = __fmul_rn(gp, n[1]); vz[c] = __fmul_rn(gp, n[2]);
                    changed = true;
                } else {  // ion charge exchange with the cold background gas
                    const float P_cx = fminf(1.0f, aa);
                    const int e = u_type < P_cx ? 1 : 0;
                    ev[c] = e | 4;
                    if (e == 0) continue;
                    uint32_t b1[4];
                    philox4x32_10(i, a.step, STREAM_COLL + (uint32_t)a.s, 1u, a.k0, a.k1, b1);
                    const float r12 = bm_r(u_a), ph12 = __fmul_rn(6.2831855f, u_b);
                    const float r3 = bm_r(u_c), ph3 = __fmul_rn(6.2831855f, u01(b1[0]));
                    vx[c] = __fmul_rn(a.gvt, __fmul_rn(r12, cosf(ph12)));
                    vy[c] = __fmul_rn(a.gvt, __fmul_rn(r12, sinf(ph12)));
                    vz[c] = __fmul_rn(a.gvt, __fmul_rn(r3, cosf(ph3)));
                    changed = true;
                }
            }
            if (changed) {
                if (i0 + 3 < n_sorted) {
                    *reinterpret_cast<float4*>(a.vx + i0) = make_float4(vx[0], vx[1], vx[2], vx[3]);
                    *reinterpret_cast<float4*>(a.vy + i0) = make_float4(vy[0], vy[1], vy[2], vy[3]);
                    *reinterpret_cast<float4*>(a.vz + i0) = make_float4(vz[0], vz[1], vz[2], vz[3]);
                } else {  // the group straddles the birth tail: never touch slots >= n_sorted
#pragma unroll
                    for (int c = 0; c < 4; ++c)
                        if (i0 + c < n_sorted) { a.vx[i0 + c] = vx[c]; a.vy[i0 + c] = vy[c]; a.vz[i0 + c] = vz[c]; }
                }
            }
        }
        if (a.mask) {
            uchar4 m = make_uchar4(ev[0] & 3, ev[1] & 3, ev[2] & 3, ev[3] & 3);
            *reinterpret_cast<uchar4*>(a.mask + i0) = m;  // mask has capacity slots, 4-aligned
        }
    }
    // event counters: warp reduce, then one shared add per warp, one global add per block
    {
        int c0 = 0, c1 = 0, c2 = 0, c3 = 0;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            if (ev[c] & 4) { const int e = ev[c] & 3; c0 += e == 0; c1 += e == 1; c2 += e == 2; c3 += e == 3; }
        }
        int vals[6] = {n_cand, c0, c1, c2, c3, n_over};
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            const int r = warp_sum(vals[q]);
            if (lane == 0 && r) atomicAdd(&s_cnt[q], (ull)r);
        }
    }
    // ordered births (electron species only): exclusive prefix of n_ion inside the block ...
    int inc = n_ion;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[wp] = inc;
    __syncthreads();
    int warp_excl = 0, nb = 0;
#pragma unroll
    for (int q = 0; q < PIC1D_NWARP; ++q) { if (q < wp) warp_excl += s_w[q]; nb += s_w[q]; }
    if (tid == 0) {
        if (s_cnt[0]) atomicAdd(&sp.n_candidates, s_cnt[0]);
#pragma unroll
        for (int q = 0; q < 4; ++q) if (s_cnt[1 + q]) atomicAdd(&sp.n_events[q], s_cnt[1 + q]);
        if (s_cnt[5]) atomicAdd(&sp.over_cap, s_cnt[5]);
    }
    if (a.kind != 1) return;
    // ... and across blocks by decoupled look-back over the tiles before this one
    if (tid == 0) {
        volatile ull* desc = a.desc;
        int excl = 0;
        if (tile == 0) {
            desc[0] = desc_pack(epoch, DESC_PREFIX, nb);
        } else {
            desc[tile] = desc_pack(epoch, DESC_AGG, nb);
            __threadfence();
            int j = tile - 1;
            while (true) {
                const ull d = desc[j];
                if ((uint32_t)(d >> 32) != epoch) continue;  // not published yet this step
                const ull flag = (d >> 30) & 3ull;
                excl += (int)(d & 0x3fffffffull);
                if (flag == DESC_PREFIX) break;
                --j;
            }
            desc[tile] = desc_pack(epoch, DESC_PREFIX, excl + nb);
        }
        __threadfence();
        s_excl = excl;
        if (tile == n_act - 1) {  // last tile: close the step's birth bookkeeping
            const int total = excl + nb;
            const int ne = st->sp[0].n_sorted;
            int room = a.cap_e - ne;
            if (a.n_species > 1) room = min(room, a.cap_i - st->sp[1].n_sorted);
            const int kept = min(total, max(room, 0));
            st->sp[0].n_live = ne + kept;
            st->sp[0].births += (ull)kept;
            if (a.n_species > 1) {
                st->sp[1].n_live = st->sp[1].n_sorted + kept;
                st->sp[1].births += (ull)kept;
            }
            if (total > kept) {
                st->sp[0].dropped += (ull)(total - kept);
                if (a.n_species > 1) st->sp[1].dropped += (ull)(total - kept);
                atomicOr(&st->err, ERRBIT_CAPACITY);
            }
        }
    }
    if (nb == 0) return;  // block-uniform
    __syncthreads();
    if (n_ion == 0) return;
    int b = s_excl + warp_excl + inc - n_ion;  // birth index of this thread's first ionisation
    const int ne = st->sp[0].n_sorted, ni = a.n_species > 1 ? st->sp[1].n_sorted : 0;
    int room = a.cap_e - ne;
    if (a.n_species > 1) room = min(room, a.cap_i - ni);
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        if ((ev[c] & 3) != 3) continue;
        if (b < room) {
            const uint32_t i = (uint32_t)(i0 + c);
            uint32_t b0[4], b1[4], b2[4];
            philox4x32_10(i, a.step, STREAM_COLL + (uint32_t)a.s, 0u, a.k0, a.k1, b0);
            philox4x32_10(i, a.step, STREAM_COLL + (uint32_t)a.s, 1u, a.k0, a.k1, b1);
            philox4x32_10(i, a.step, STREAM_COLL + (uint32_t)a.s, 2u, a.k0, a.k1, b2);
            const float xp = a.x[i];
            float n2[3];
            iso_dir(u01(b0[3]), u01(b1[0]), n2);
            const float gp = gp_ion[c];
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
        ++b;
    }
}
