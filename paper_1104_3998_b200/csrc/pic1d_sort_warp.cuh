// pic1d_sort_warp.cuh -- the fine sort for species that obey Eq. 5 ("only a small
// number of particles leaves its sorting cell during one time step"): ions always, electrons of
// Courant-respecting runs.
//
// Same two passes and the same pool / bin-scan bookkeeping as pic1d_sort.cuh, but a tile is the 256
// consecutive slots ONE WARP owns, so no pass contains a block barrier: 32 independent warps per SM
// stream through the particles and hide each other's latencies.
//
//   pass 1  k_push_count_w    x, vx -> push -> key; window [lo, hi] by redux; histogram of the warp's
//                             256 keys in a 32-counter shared row (red.shared); fixed pool row of 32 bins
//   pass 2  k_push_scatter_w  identical push; lane b keeps the next free destination of window bin b in
//                             a shared row; per row of 32 slots: match.any groups equal keys, the lowest
//                             lane of a group reads and advances the bin's cursor, the others take
//                             cursor + (number of lower lanes with the same key).  Rows are taken in
//                             slot order, so the sort is stable (R18) and no atomic is used.
// Tiles whose window is wider than 32 bins (a species' birth tail, fast sheath ions) take a pool row
// from the overflow region and keep their cursors in that row in global memory: slower, rare.
#pragma once
#include "pic1d_sort.cuh"

#define PIC1D_TW 256  // slots per warp tile
#define PIC1D_PSW 32  // bins of the fixed pool row of a warp tile (= warp size: lane b <-> window bin b)

template <int BC>
__global__ void __launch_bounds__(PIC1D_NT) k_push_count_w(SortArgs a) {
    __shared__ int s_h[PIC1D_NWARP][PIC1D_PSW + 1];  // + a slot that swallows the keys outside the window (never read)
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    DevSpecies& sp = a.st->sp[a.s];
    const int n_tiles = sp.n_tiles, n_src = sp.n_src, n_push = sp.n_push;
    const int n_warps = gridDim.x * PIC1D_NWARP;
    const uint32_t step = a.st->step;
    int n_refl = 0;
    for (int tile = blockIdx.x * PIC1D_NWARP + wp; tile < n_tiles; tile += n_warps) {
        const int base = tile * PIC1D_TW;
        int keys[8];
        unsigned ulo = 0xffffffffu;
        int hi = -1, smin = 0;
        bool nonfinite = false;
        const bool full = base + PIC1D_TW <= n_push && a.keys_dbg == nullptr;  // warp-uniform
        if (full) {
            float4 X[2], VX[2];
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                const int idx = base + v * 128 + lane * 4;
                X[v] = __ldcs(reinterpret_cast<const float4*>(a.sx + idx));
                VX[v] = __ldcs(reinterpret_cast<const float4*>(a.svx + idx));
            }
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                float xs[4] = {X[v].x, X[v].y, X[v].z, X[v].w}, vs[4] = {VX[v].x, VX[v].y, VX[v].z, VX[v].w};
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int key = push_particle<BC>(xs[c], vs[c], true, a.E32, a.kappa, a.Nc, a.fNc, a.inv_r, a.shift, a.rp, step, (unsigned)(base + v * 128 + lane * 4 + c), n_refl);
                    ulo = min(ulo, (unsigned)key); hi = max(hi, key); smin = min(smin, key);
                    if (key == -2) nonfinite |= (xs[c] != xs[c]);
                    keys[v * 4 + c] = key;
                }
            }
        } else {
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                const int idx = base + v * 128 + lane * 4;
                float4 X = make_float4(0.f, 0.f, 0.f, 0.f), VX = X;
                if (idx < n_src) {
                    X = __ldcs(reinterpret_cast<const float4*>(a.sx + idx));
                    VX = __ldcs(reinterpret_cast<const float4*>(a.svx + idx));
                }
                float xs[4] = {X.x, X.y, X.z, X.w}, vs[4] = {VX.x, VX.y, VX.z, VX.w};
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int i = idx + c;
                    int key = -3;  // no particle
                    smin = min(smin, i < n_src ? 0 : -3);
                    if (i < n_src) {
                        key = push_particle<BC>(xs[c], vs[c], i < n_push, a.E32, a.kappa, a.Nc, a.fNc, a.inv_r, a.shift, a.rp, step, (unsigned)i, n_refl);
                        ulo = min(ulo, (unsigned)key); hi = max(hi, key); smin = min(smin, key);
                        if (key == -2) nonfinite |= (xs[c] != xs[c]);
                        if (a.keys_dbg) a.keys_dbg[i] = key >= 0 ? key : -1;
                    }
                    keys[v * 4 + c] = key;
                }
            }
        }
        ulo = __reduce_min_sync(0xffffffffu, ulo); hi = __reduce_max_sync(0xffffffffu, hi);
        int lo = (int)ulo, dl = 0, dr = 0;
        if (__any_sync(0xffffffffu, smin < 0)) {  // an absorbed or missing particle in the tile: rare
            int lo2 = 0x7fffffff;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                dl += keys[q] == -1; dr += keys[q] == -2;
                if (keys[q] >= 0) lo2 = min(lo2, keys[q]);
            }
            dl = __reduce_add_sync(0xffffffffu, dl); dr = __reduce_add_sync(0xffffffffu, dr);
            lo = __reduce_min_sync(0xffffffffu, lo2);
        }
        if (nonfinite) atomicOr(&a.st->err, ERRBIT_NONFINITE);
        const int w = hi >= 0 ? hi - lo + 1 : 0;
        if (w == 0) lo = 0;
        int off = tile * PIC1D_PSW;
        if (w > PIC1D_PSW) {  // overflow region
            int o = 0;
            if (lane == 0) {
                o = atomicAdd(&sp.pool_used, w);
                if (o + w > a.pool_size - a.pool_fixed) { o = -1; atomicOr(&a.st->err, ERRBIT_WORKSPACE); }
            }
            o = __shfl_sync(0xffffffffu, o, 0);
            off = o >= 0 ? a.pool_fixed + o : -1;
        }
        if (lane == 0) {
            if (w > 0) {
                atomicMin(&a.grp_lo[tile / PIC1D_GROUP], lo);
                atomicMax(&a.grp_hi[tile / PIC1D_GROUP], hi);
            }
            a.tile_lo[tile] = lo; a.tile_w[tile] = off >= 0 ? w : 0; a.tile_off[tile] = off;
            a.tile_dead[tile] = dl + dr;
            if (off < 0) atomicAdd(&sp.dropped, (ull)(min(PIC1D_TW, n_src - base) - dl - dr));  // the tile is lost (sticky error)
            if (dl) atomicAdd(&sp.absorbed_left, (ull)dl);
            if (dr) atomicAdd(&sp.absorbed_right, (ull)dr);
        }
        if (w <= PIC1D_PSW) {
            // histogram of the warp's keys in a 32-counter shared row
            s_h[wp][lane] = 0;
            __syncwarp();
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const unsigned r = (unsigned)(keys[q] - lo);  // absorbed: huge
                atomicAdd(&s_h[wp][min(r, (unsigned)PIC1D_PSW)], 1);  // branch-free
            }
            __syncwarp();
            if (lane < w) a.pool[off + lane] = s_h[wp][lane];
            __syncwarp();
        } else if (off >= 0) {
            // wide window (rare): zero the tile's overflow row, then count straight into it
            for (int i = lane; i < w; i += 32) a.pool[off + i] = 0;
            __threadfence();
            __syncwarp();
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (keys[q] >= 0) atomicAdd(&a.pool[off + keys[q] - lo], 1);
        }
    }
    if (a.rp.prob > 0.0f) {  // reflections are counted here only (the scatter repeats the same decisions)
        n_refl = __reduce_add_sync(0xffffffffu, n_refl);
        if (lane == 0 && n_refl) atomicAdd(&sp.reflected, (ull)n_refl);
    }
}

// MCCK != 0: the species' null-collision MCC is folded in (mcc_lane: the destination slot is the particle id)
template <int BC, bool ABS, int MCCK>
__global__ void __launch_bounds__(PIC1D_NT, 4) k_push_scatter_w(SortArgs a) {
    __shared__ unsigned s_cur[PIC1D_NWARP][PIC1D_PSW + 1];  // next free destination per window bin (+ absorbed)
    constexpr int ROWS = PIC1D_TW / 32;
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    DevSpecies& sp = a.st->sp[a.s];
    const int n_tiles = sp.n_tiles, n_src = sp.n_src, n_push = sp.n_push;
    const int n_warps = gridDim.x * PIC1D_NWARP;
    unsigned* cur = s_cur[wp];
    const uint32_t step = a.st->step;
    int n_refl = 0;  // (counted by the counting pass)
    MccCount mc = {0u, 0u, 0u};
    for (int tile = blockIdx.x * PIC1D_NWARP + wp; tile < n_tiles; tile += n_warps) {
        const int lo = a.tile_lo[tile], w = a.tile_w[tile], off = a.tile_off[tile];
        if (off < 0) continue;  // count pool exhausted (sticky error): the tile is lost (counted by the counting pass)
        const int base = tile * PIC1D_TW + lane;
        const bool full = tile * PIC1D_TW + PIC1D_TW <= n_push;  // warp-uniform
        const bool narrow = w <= PIC1D_PSW;
        float x[ROWS], vx[ROWS], vy[ROWS], vz[ROWS];
        int k[ROWS];  // bin relative to the window; w = absorbed (ABS); -1 = no particle; MCCK: then the destination
        unsigned wall = 0;
        if (full) {
#pragma unroll
            for (int r = 0; r < ROWS; ++r) { x[r] = __ldcs(a.sx + base + r * 32); vx[r] = __ldcs(a.svx + base + r * 32); }
        } else {
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const int i = base + r * 32;
                x[r] = 0.0f; vx[r] = 0.0f;
                if (i < n_src) { x[r] = __ldcs(a.sx + i); vx[r] = __ldcs(a.svx + i); }
            }
        }
        // cursors of the window bins: first destination of this tile's particles per bin
        unsigned c0 = 0;
        if (narrow && lane < w) c0 = (unsigned)(a.offsets[lo + lane] + __ldcg(a.pool + off + lane));
        unsigned cdead = 0;
        if (ABS) cdead = (unsigned)a.tile_dead[tile];  // prefix inside the tile's chunk of the absorbed-count scan
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
            const int i = base + r * 32;
            k[r] = -1;
            if (full || i < n_src) {
                const int key = push_particle<BC>(x[r], vx[r], full || i < n_push, a.E32, a.kappa, a.Nc, a.fNc, a.inv_r, a.shift, a.rp, step, (unsigned)i, n_refl);
                k[r] = key >= 0 ? key - lo : (ABS ? w : -1);
                if (ABS && key == -2) wall |= 1u << r;
            }
        }
        if (ABS) {  // rare: the tile lost particles to a wall -> its place in the ordered absorbed list needs the chunk's base
            bool dead = false;
#pragma unroll
            for (int r = 0; r < ROWS; ++r) dead |= k[r] == w;
            if (__any_sync(0xffffffffu, dead)) cdead += (unsigned)sp.dead_base[tile / dead_chunk_tiles(n_tiles)];
        }
        if (full) {
#pragma unroll
            for (int r = 0; r < ROWS; ++r) { vy[r] = __ldcs(a.svy + base + r * 32); vz[r] = __ldcs(a.svz + base + r * 32); }
        } else {
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const int i = base + r * 32;
                vy[r] = 0.0f; vz[r] = 0.0f;
                if (i < n_src) { vy[r] = __ldcs(a.svy + i); vz[r] = __ldcs(a.svz + i); }
            }
        }
        __syncwarp();  // the previous tile's rows are done with the cursors
        if (narrow) {
            cur[lane] = lane < w ? c0 : cdead;     // bin w (the absorbed pseudo-bin, ABS) follows the window
            if (lane == 0) cur[PIC1D_PSW] = cdead;  // ... also when the window has all 32 bins
            __syncwarp();
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const int kk = k[r];
                const unsigned peers = __match_any_sync(0xffffffffu, kk);
                const int leader = __ffs(peers) - 1;
                unsigned old = 0;
                if (kk >= 0 && lane == leader) { old = cur[kk]; cur[kk] = old + __popc(peers); }
                old = __shfl_sync(0xffffffffu, old, leader);
                const unsigned d = old + __popc(peers & lanemask_lt());
                if (kk >= 0) {
                    if (!ABS || kk < w) {
                        if (!MCCK) { a.dx[d] = x[r]; a.dvx[d] = vx[r]; a.dvy[d] = vy[r]; a.dvz[d] = vz[r]; }
                        else k[r] = (int)d | (1 << 30);  // remember the slot (= particle id); stored below
                    } else {
                        if (a.abs_list && (int)d < a.abs_cap)  // absorbed: ordered list of (slot, wall)
                            a.abs_list[d] = (unsigned)(base + r * 32) | (((wall >> r) & 1u) << 31);
                        if (MCCK) k[r] = -1;
                    }
                }
                __syncwarp();  // the next row's leaders see the advanced cursors
            }
        } else {
            // wide window: the cursors stay in the tile's pool row (exclusive prefixes over earlier tiles)
            if (ABS && lane == 0) cur[0] = cdead;
            __syncwarp();
            volatile int* row = a.pool + off;
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const int kk = k[r];
                const unsigned peers = __match_any_sync(0xffffffffu, kk);
                const int leader = __ffs(peers) - 1;
                unsigned old = 0;
                if (kk >= 0 && lane == leader) {
                    if (!ABS || kk < w) { old = (unsigned)row[kk]; row[kk] = (int)(old + __popc(peers)); old += (unsigned)a.offsets[lo + kk]; }
                    else { old = cur[0]; cur[0] = old + __popc(peers); }
                }
                old = __shfl_sync(0xffffffffu, old, leader);
                const unsigned d = old + __popc(peers & lanemask_lt());
                if (kk >= 0) {
                    if (!ABS || kk < w) {
                        if (!MCCK) { a.dx[d] = x[r]; a.dvx[d] = vx[r]; a.dvy[d] = vy[r]; a.dvz[d] = vz[r]; }
                        else k[r] = (int)d | (1 << 30);
                    } else {
                        if (a.abs_list && (int)d < a.abs_cap)
                            a.abs_list[d] = (unsigned)(base + r * 32) | (((wall >> r) & 1u) << 31);
                        if (MCCK) k[r] = -1;
                    }
                }
                __syncwarp();
            }
        }
        if (MCCK) {
            // All destinations are known: the stores and the null-test look-ups of the 8 rows go out together.
            unsigned nw[ROWS];
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                nw[r] = 0u;
                if (k[r] >= 0) {
                    const unsigned d = (unsigned)k[r] & 0x3fffffffu;
                    k[r] = (int)d;
                    a.dx[d] = x[r]; a.dvx[d] = vx[r]; a.dvy[d] = vy[r]; a.dvz[d] = vz[r];
                    nw[r] = __ldcg(a.m.null_bits + (d >> 5));
                    if (a.m.mask) a.m.mask[d] = 0;
                }
            }
            unsigned cmask = 0;  // rows whose particle passed the null test
#pragma unroll
            for (int r = 0; r < ROWS; ++r)
                if (k[r] >= 0 && ((nw[r] >> ((unsigned)k[r] & 31u)) & 1u)) cmask |= 1u << r;
            // The tile's candidates (few: P0 of the particles), one per lane and round: selection,
            // kinematics, and the collided velocity overwrites the one this lane has just stored.
            while (__any_sync(0xffffffffu, cmask != 0u)) {
                const bool has = cmask != 0u;
                const int r = has ? __ffs(cmask) - 1 : 0;
                cmask &= cmask - 1u;
                unsigned d = 0;
                float cx = 0.0f, cy = 0.0f, cz = 0.0f;
#pragma unroll
                for (int q = 0; q < ROWS; ++q)
                    if (q == r) { d = (unsigned)k[q]; cx = vx[q]; cy = vy[q]; cz = vz[q]; }
                const int e = mcc_lane<MCCK>(a.m, step, d, has, cx, cy, cz, mc);
                if (e) {
                    a.dvx[d] = cx; a.dvy[d] = cy; a.dvz[d] = cz;
                    if (a.m.mask) a.m.mask[d] = (uint8_t)e;
                }
            }
        }
    }
    if (MCCK) mcc_flush_counts(a.m, mc);
}
