// pic1d_sort.cuh -- fused gather + push + boundary with the fine sort.
//
// The paper sorts in place with per-cell slack and shared/global atomic counters (L166-186); here
// the sort is a compact, STABLE counting sort in two passes over the particles, and the push is
// recomputed in the second pass instead of being stored in between:
//
//   pass 1  k_push_count    read x, vx (8 B/particle); push; boundary; key; per-tile histogram in
//                           shared memory; the tile's window [lo, hi] of counts goes to a pool
//   scan    k_bin_scan      per sort cell k: exclusive prefix over tiles of count[t][k] (in place),
//                           total -> hist[k]; the last block to finish scans hist -> offsets[N_sc + 1]
//                           (+ 64 extra blocks: chunked prefix of the per-tile absorbed counts; + blocks that
//                           compute a folded species' null-test mask when it was not computed one step ahead)
//   pass 2  k_push_scatter  read x, vx, vy, vz (16 B); identical push; stable rank inside the tile
//                           (warp-private shared counters, warps in order); write the four arrays to
//                           offsets[k] + prefix[t][k] + rank (16 B), through a tile-sorted shared-memory
//                           staging buffer when the tile spreads over many cells
//
// A tile is T consecutive source slots.  Because the source is sorted by last step's cell, a tile's
// keys fall in a narrow window when particles move about one cell per step (Eq. 5); nothing
// breaks when they do not (configs 2-4 electrons), the window just gets wider.
#pragma once
#include "pic1d_device.cuh"
#include "pic1d_mcc.cuh"

struct SortArgs {
    const float *sx, *svx, *svy, *svz;  // source buffer
    float *dx, *dvx, *dvy, *dvz;        // destination buffer
    const float* E32;
    DevState* st;
    int s;
    int *tile_lo, *tile_w, *tile_off, *tile_dead;  // per tile: window start, width, pool offset, absorbed
    int *grp_lo, *grp_hi;                          // per tile group: union window
    int* pool;
    int pool_size;    // fixed rows + overflow region
    int pool_stride;  // bins per fixed pool row (one row per tile)
    int pool_fixed;   // n_tiles_max * pool_stride: start of the overflow region
    int* hist;     // [n_sc]
    int* offsets;  // [n_sc + 1]
    int* keys_dbg; // optional, per source slot
    unsigned* abs_list;  // optional ordered list of absorbed slots (ions, for secondary emission)
    int abs_cap;
    float kappa, fNc, inv_r;
    int Nc, n_sc;
    int shift;  // key = sort cell >> shift (0 except in the coarse pass of an unsorted load)
    int WA;     // sub-window (bins) the scatter kernel ranks at a time in shared memory (a multiple of 8)
    MccP m;     // collision model of the species, for the scatter kernels that fold the MCC in
    ReflP rp;        // electron reflection at the walls (prob = 0: off)
    int null_first;  // k_bin_scan: blocks from (bin blocks + null_first) on compute the null-test bit mask
};

// ---- pass 1 -----------------------------------------------------------------------------------
// V float4 loads per thread: tile T = NT * 4 * V slots.  The tile's histogram lives in a shared
// window of WA counters relative to the tile's lowest key; wider windows are counted WA bins at a time.
// A tile whose window fits pool_stride bins owns the fixed pool row tile * pool_stride (no allocation);
// wider ones (a species' birth tail) take space from the overflow region with one atomicAdd per tile --
// the position in the pool carries no meaning, so this atomic decides no particle index.
template <int BC, int V>
__global__ void __launch_bounds__(PIC1D_NT) k_push_count(SortArgs a) {
    extern __shared__ int s_hist[];  // WA counters, all zero between tiles (+ one slot for keys outside the sub-window)
    __shared__ int s_lohi[2][2];     // block min / max of the keys, double-buffered over tiles
    __shared__ int s_dead[2][2];     // absorbed left / right, double-buffered
    __shared__ int s_off;
    constexpr int T = PIC1D_NT * 4 * V;
    const int tid = threadIdx.x, lane = tid & 31;
    const int WA = a.WA;
    DevSpecies& sp = a.st->sp[a.s];
    const int n_tiles = sp.n_tiles, n_src = sp.n_src, n_push = sp.n_push;
    const uint32_t step = a.st->step;
    int n_refl = 0;
    for (int i = tid; i < WA; i += PIC1D_NT) s_hist[i] = 0;
    if (tid < 2) { s_lohi[tid][0] = 0x7fffffff; s_lohi[tid][1] = -1; s_dead[tid][0] = 0; s_dead[tid][1] = 0; }
    __syncthreads();
    int par = 0;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, par ^= 1) {
        const int base = tile * T;
        int keys[4 * V];
        unsigned ulo = 0xffffffffu;  // absorbed keys are negative: huge as unsigned, below every max as signed
        int hi = -1, smin = 0;       // smin < 0: the thread saw an absorbed (or missing) particle
        bool nonfinite = false;
        const bool full = base + T <= n_push && a.keys_dbg == nullptr;  // block-uniform fast path
        if (full) {
            float4 X[V], VX[V];
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const int idx = base + (v * PIC1D_NT + tid) * 4;
                X[v] = __ldcs(reinterpret_cast<const float4*>(a.sx + idx));
                VX[v] = __ldcs(reinterpret_cast<const float4*>(a.svx + idx));
            }
#pragma unroll
            for (int v = 0; v < V; ++v) {
                float xs[4] = {X[v].x, X[v].y, X[v].z, X[v].w}, vs[4] = {VX[v].x, VX[v].y, VX[v].z, VX[v].w};
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int key = push_particle<BC>(xs[c], vs[c], true, a.E32, a.kappa, a.Nc, a.fNc, a.inv_r, a.shift, a.rp, step, (unsigned)(base + (v * PIC1D_NT + tid) * 4 + c), n_refl);
                    ulo = min(ulo, (unsigned)key); hi = max(hi, key); smin = min(smin, key);
                    if (key == -2) nonfinite |= (xs[c] != xs[c]);
                    keys[v * 4 + c] = key;
                }
            }
        } else {
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const int idx = base + (v * PIC1D_NT + tid) * 4;
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
        if (lane == 0) {
            if ((int)ulo >= 0) atomicMin(&s_lohi[par][0], (int)ulo);  // a warp of absorbed particles has none
            atomicMax(&s_lohi[par][1], hi);
        }
        if (__any_sync(0xffffffffu, smin < 0)) {  // some lane of the warp saw an absorbed (or missing) particle: rare
            int ndl = 0, ndr = 0;
            int lo2 = 0x7fffffff;
#pragma unroll
            for (int q = 0; q < 4 * V; ++q) {
                ndl += keys[q] == -1; ndr += keys[q] == -2;
                if (keys[q] >= 0) lo2 = min(lo2, keys[q]);
            }
            ndl = __reduce_add_sync(0xffffffffu, ndl); ndr = __reduce_add_sync(0xffffffffu, ndr);
            lo2 = __reduce_min_sync(0xffffffffu, lo2);
            if (lane == 0) {
                if (ndl) atomicAdd(&s_dead[par][0], ndl);
                if (ndr) atomicAdd(&s_dead[par][1], ndr);
                if (lo2 != 0x7fffffff) atomicMin(&s_lohi[par][0], lo2);
            }
        }
        if (nonfinite) atomicOr(&a.st->err, ERRBIT_NONFINITE);
        __syncthreads();
        const int L0 = s_lohi[par][0], H = s_lohi[par][1];
        const int w = H >= L0 ? H - L0 + 1 : 0;
        const int lo = w > 0 ? L0 : 0;
        int off = tile * a.pool_stride;
        if (w > a.pool_stride) {  // block-uniform; overflow region
            if (tid == 0) {
                int o = atomicAdd(&sp.pool_used, w);
                if (o + w > a.pool_size - a.pool_fixed) { o = -1; atomicOr(&a.st->err, ERRBIT_WORKSPACE); }
                s_off = o >= 0 ? a.pool_fixed + o : -1;
            }
            __syncthreads();
            off = s_off;
        }
        if (tid == 0) {
            const int dl = s_dead[par][0], dr = s_dead[par][1];
            if (w > 0) {
                atomicMin(&a.grp_lo[tile / PIC1D_GROUP], lo);
                atomicMax(&a.grp_hi[tile / PIC1D_GROUP], H);
            }
            a.tile_lo[tile] = lo; a.tile_w[tile] = off >= 0 ? w : 0; a.tile_off[tile] = off;
            a.tile_dead[tile] = dl + dr;
            if (off < 0) atomicAdd(&sp.dropped, (ull)(min(T, n_src - base) - dl - dr));  // the tile is lost (sticky error)
            if (dl) atomicAdd(&sp.absorbed_left, (ull)dl);
            if (dr) atomicAdd(&sp.absorbed_right, (ull)dr);
            // reset the OTHER buffer for the next tile (nobody touches it before the next barrier)
            s_lohi[par ^ 1][0] = 0x7fffffff; s_lohi[par ^ 1][1] = -1; s_dead[par ^ 1][0] = 0; s_dead[par ^ 1][1] = 0;
        }
        for (int sub = 0; sub < w; sub += WA) {
            const int nsub = min(WA, w - sub), klo = lo + sub;
            // histogram: one shared-memory reduction per particle (conflicting red.shared is not
            // serialised on sm_100a: 3 cycles per warp instruction)
#pragma unroll
            for (int q = 0; q < 4 * V; ++q) {
                const unsigned r = (unsigned)(keys[q] - klo);
                atomicAdd(&s_hist[r < (unsigned)nsub ? r : (unsigned)WA], 1);  // branch-free: slot WA swallows the rest (never read)
            }
            __syncthreads();
            for (int i = tid; i < nsub; i += PIC1D_NT) {
                if (off >= 0) a.pool[off + sub + i] = s_hist[i];
                s_hist[i] = 0;
            }
            __syncthreads();
        }
        if (w == 0) __syncthreads();  // keep the double buffer two barriers apart
    }
    if (a.rp.prob > 0.0f) {  // reflections are counted here only (the scatter repeats the same decisions)
        n_refl = __reduce_add_sync(0xffffffffu, n_refl);
        if (lane == 0 && n_refl) atomicAdd(&sp.reflected, (ull)n_refl);
    }
}

// block-wide exclusive scan of src[0..n) into dst[0..n), returns the total; single block, any n.
// Every warp owns a contiguous segment and walks it in rows of 32 (coalesced): pass 1 sums the
// segment (independent loads), a shuffle scan orders the warps, pass 2 scans row by row with a carry.
// dst may alias src.
// SPARSE: rows of 32 zeros are skipped (their dst entries are NOT written: callers only read the
// prefix at positions whose src was non-zero).
template <bool SPARSE = false>
__device__ int block_exclusive_scan(const int* src, int* dst, int n) {
    __shared__ int s_w[33];
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5, nw = blockDim.x >> 5;
    const int seg = ((n + nw * 32 - 1) / (nw * 32)) * 32;  // elements per warp, a multiple of 32
    const int b = min(wp * seg, n), e = min(b + seg, n);
    int tot = 0;
    for (int i = b + lane; i < e; i += 32 * 8) {
        int v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = i + u * 32 < e ? __ldcg(src + i + u * 32) : 0;
#pragma unroll
        for (int u = 0; u < 8; ++u) tot += v[u];
    }
    tot = __reduce_add_sync(0xffffffffu, tot);
    __syncthreads();  // s_w may still be read by a previous call
    if (lane == 0) s_w[wp] = tot;
    __syncthreads();
    if (wp == 0) {
        const int t = lane < nw ? s_w[lane] : 0;
        int ti = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, ti, o);
            if (lane >= o) ti += u;
        }
        s_w[lane] = ti - t;  // exclusive over warps
        if (lane == 31) s_w[32] = ti;
    }
    __syncthreads();
    int carry = s_w[wp];
    for (int i0 = b; i0 < e; i0 += 32 * 4) {
        int v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = i0 + u * 32 + lane < e ? __ldcg(src + i0 + u * 32 + lane) : 0;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (SPARSE && !__any_sync(0xffffffffu, v[u] != 0)) continue;
            int inc = v[u];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (i0 + u * 32 + lane < e) dst[i0 + u * 32 + lane] = carry + inc - v[u];
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
    return s_w[32];
}

// ---- scan over tiles, per sort cell --------------------------------------------------------------
// Block = 32 adjacent sort cells (lane = cell k) x 32 warps.  The tiles whose window can contain the
// block's cells form a short range [ta, tb) (found from the tile-group windows); it is split evenly
// over the warps.  Pass 1 sums each warp's share, a shared-memory prefix orders the warps, pass 2
// rewrites pool[tile_off[t] + k - tile_lo[t]] as the number of particles of tiles < t with key k
// (exclusive prefix over tiles); hist[k] gets the total.  Row segments of the pool are read coalesced.
// The bin block that finishes last turns the histogram into offsets[k] = #{key < k} and closes the sort's
// counts (n_live = n_sorted = survivors): the former k_offsets_scan, saved as a launch.
__device__ void bin_scan_finish(const SortArgs& a) {
    __shared__ int s_last;
    DevSpecies& sp = a.st->sp[a.s];
    __syncthreads();  // this block's hist entries are written
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(&sp.scan_done, 1) == (a.n_sc + 31) / 32 - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int total = block_exclusive_scan<false>(a.hist, a.offsets, a.n_sc);
    if (threadIdx.x == 0) {
        a.offsets[a.n_sc] = total;
        sp.n_live = total;
        sp.n_sorted = total;
    }
}

// NW warps per block: 16 (with 16 tiles in flight per warp the best of the sweep in profiles/r2_notes.md) when the bin
// blocks alone fill the GPU or the problem is small, 32 when few bin blocks walk many tiles (coarse sort cells: 8
// blocks for config 3 at r = 16)
#define BINSCAN_B 16   // tiles in flight per warp
#define BINSCAN_LIST 4096
#define BINSCAN_DESC 2048  // tile descriptors a block can keep in shared memory
template <int NW>
__global__ void __launch_bounds__(NW * 32) k_bin_scan(SortArgs a) {
    __shared__ int s_wc[NW];
    __shared__ unsigned short s_list[BINSCAN_LIST];  // tile groups whose window overlaps the block's cells
    __shared__ int s_part[NW][33];
    __shared__ int4 s_desc[BINSCAN_DESC];
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    const int nb_bins = (a.n_sc + 31) / 32;
    if ((int)blockIdx.x >= nb_bins + a.null_first) {
        // extra blocks (species whose MCC is folded into the scatter): the null-test bit mask of this step,
        // 1024 words = 32768 slots per block, concurrently with the bin blocks
        mcc_null_words(a.m, ((int)blockIdx.x - nb_bins - a.null_first) * (NW * 32) + tid);
        return;
    }
    if ((int)blockIdx.x >= nb_bins) {
        // PIC1D_DEAD_CHUNKS extra blocks (species with an ordered absorbed list only), concurrently with the bin
        // blocks: exclusive prefix of the per-tile absorbed counts inside the block's chunk of tiles; the block
        // that finishes last turns the chunk totals into chunk bases (the scatter adds base + prefix).  One block
        // scanning all 2.7e5 warp tiles of config 4 took 70 us and bounded the whole launch.
        __shared__ int s_last_dead;
        DevSpecies& sp = a.st->sp[a.s];
        const int c = (int)blockIdx.x - nb_bins, ch = dead_chunk_tiles(sp.n_tiles);
        const int b = min(c * ch, sp.n_tiles), e = min(b + ch, sp.n_tiles);
        const int tot = block_exclusive_scan<true>(a.tile_dead + b, a.tile_dead + b, e - b);
        if (tid == 0) {
            sp.dead_tot[c] = tot;
            __threadfence();
            s_last_dead = atomicAdd(&sp.dead_done, 1) == PIC1D_DEAD_CHUNKS - 1;
        }
        __syncthreads();
        if (s_last_dead && tid == 0) {
            __threadfence();
            int run = 0;
            for (int q = 0; q < PIC1D_DEAD_CHUNKS; ++q) {
                sp.dead_base[q] = run;
                run += *reinterpret_cast<volatile int*>(&sp.dead_tot[q]);
            }
            sp.n_dead = run;
        }
        return;
    }
    const int kb0 = blockIdx.x * 32, kb1 = min(kb0 + 31, a.n_sc - 1);
    const int k = kb0 + lane;
    const int n_tiles = a.st->sp[a.s].n_tiles;
    const int n_groups = (n_tiles + PIC1D_GROUP - 1) / PIC1D_GROUP;
    // ordered list of the relevant groups (a group is skipped as a whole: the birth tail of a species
    // has full-width windows and must not drag every tile before it into the walk).  Thread t owns the
    // contiguous chunk of groups [t gpt, (t+1) gpt): count, block-wide exclusive scan, write.
    int n_rel = 0;
    {
        const int gpt = (n_groups + NW * 32 - 1) / (NW * 32);
        const int g_beg = min(tid * gpt, n_groups), g_end = min(g_beg + gpt, n_groups);
        int mine = 0;
        for (int g = g_beg; g < g_end; ++g) mine += (a.grp_hi[g] >= kb0 && a.grp_lo[g] <= kb1) ? 1 : 0;
        int inc = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_wc[wp] = inc;
        __syncthreads();
        int before = 0;
#pragma unroll 8
        for (int q = 0; q < NW; ++q) { const int v = s_wc[q]; if (q < wp) before += v; n_rel += v; }
        int idx = before + inc - mine;
        if (mine) {
            for (int g = g_beg; g < g_end; ++g)
                if (a.grp_hi[g] >= kb0 && a.grp_lo[g] <= kb1) { if (idx < BINSCAN_LIST) s_list[idx] = (unsigned short)g; ++idx; }
        }
        __syncthreads();
    }
    // n_rel groups (or, if the list overflowed, every group) -> virtual tile range split over the warps
    const bool listed = n_rel <= BINSCAN_LIST && n_groups <= 65536;
    const int n_virt = (listed ? n_rel : n_groups) * PIC1D_GROUP;
    const int chunk = (n_virt + NW - 1) / NW;
    const int v_beg = min(wp * chunk, n_virt), v_end = min(v_beg + chunk, n_virt);
    constexpr int B = BINSCAN_B;  // tiles in flight per warp: the loads of a batch are independent
    if (listed && n_virt <= BINSCAN_DESC) {
        // usual case: the descriptors (lo, w, off) of the listed tiles are fetched once, coalesced, into
        // shared memory; both passes then read them with one broadcast LDS.128 and no index arithmetic
        for (int v = tid; v < n_virt; v += NW * 32) {
            const int t = (int)s_list[v / PIC1D_GROUP] * PIC1D_GROUP + v % PIC1D_GROUP;
            s_desc[v] = t < n_tiles ? make_int4(a.tile_lo[t], a.tile_w[t], a.tile_off[t], 0) : make_int4(0, 0, 0, 0);
        }
        __syncthreads();
        int sum = 0;
        for (int v0 = v_beg; v0 < v_end; v0 += B) {
            int c[B];
#pragma unroll
            for (int b = 0; b < B; ++b) {
                c[b] = 0;
                if (v0 + b < v_end) {
                    const int4 d = s_desc[v0 + b];
                    const unsigned r = (unsigned)(k - d.x);
                    if (r < (unsigned)d.y) c[b] = __ldcg(a.pool + d.z + r);
                }
            }
#pragma unroll
            for (int b = 0; b < B; ++b) sum += c[b];
        }
        s_part[wp][lane] = sum;
        __syncthreads();
        int run = 0, total = 0;
#pragma unroll 8
        for (int q = 0; q < NW; ++q) {
            const int v = s_part[q][lane];
            if (q < wp) run += v;
            total += v;
        }
        for (int v0 = v_beg; v0 < v_end; v0 += B) {
            int p[B];  // index into the pool, -1: the tile's window does not hold the cell
            int c[B];
#pragma unroll
            for (int b = 0; b < B; ++b) {
                p[b] = -1;
                c[b] = 0;
                if (v0 + b < v_end) {
                    const int4 d = s_desc[v0 + b];
                    const unsigned r = (unsigned)(k - d.x);
                    if (r < (unsigned)d.y) p[b] = d.z + (int)r;
                }
            }
#pragma unroll
            for (int b = 0; b < B; ++b) if (p[b] >= 0) c[b] = __ldcg(a.pool + p[b]);
#pragma unroll
            for (int b = 0; b < B; ++b) if (p[b] >= 0) { __stcg(a.pool + p[b], run); run += c[b]; }
        }
        if (wp == 0 && k < a.n_sc) a.hist[k] = total;
        bin_scan_finish(a);
        return;
    }
    int sum = 0;
    for (int v0 = v_beg; v0 < v_end; v0 += B) {
        int c[B];
#pragma unroll
        for (int b = 0; b < B; ++b) {
            c[b] = 0;
            const int v = v0 + b;
            if (v < v_end) {
                const int t = (listed ? (int)s_list[v / PIC1D_GROUP] : v / PIC1D_GROUP) * PIC1D_GROUP + v % PIC1D_GROUP;
                if (t < n_tiles) {
                    const unsigned r = (unsigned)(k - a.tile_lo[t]);
                    if (r < (unsigned)a.tile_w[t]) c[b] = __ldcg(a.pool + a.tile_off[t] + r);
                }
            }
        }
#pragma unroll
        for (int b = 0; b < B; ++b) sum += c[b];
    }
    s_part[wp][lane] = sum;
    __syncthreads();
    int run = 0, total = 0;
#pragma unroll 8
    for (int q = 0; q < NW; ++q) {
        const int v = s_part[q][lane];
        if (q < wp) run += v;
        total += v;
    }
    for (int v0 = v_beg; v0 < v_end; v0 += B) {
        int* p[B];
        int c[B];
#pragma unroll
        for (int b = 0; b < B; ++b) {
            p[b] = nullptr;
            c[b] = 0;
            const int v = v0 + b;
            if (v < v_end) {
                const int t = (listed ? (int)s_list[v / PIC1D_GROUP] : v / PIC1D_GROUP) * PIC1D_GROUP + v % PIC1D_GROUP;
                if (t < n_tiles) {
                    const unsigned r = (unsigned)(k - a.tile_lo[t]);
                    if (r < (unsigned)a.tile_w[t]) p[b] = a.pool + a.tile_off[t] + r;
                }
            }
        }
#pragma unroll
        for (int b = 0; b < B; ++b) if (p[b]) c[b] = __ldcg(p[b]);
#pragma unroll
        for (int b = 0; b < B; ++b) if (p[b]) { __stcg(p[b], run); run += c[b]; }
    }
    if (wp == 0 && k < a.n_sc) a.hist[k] = total;
    bin_scan_finish(a);
}

// ---- pass 2 -----------------------------------------------------------------------------------
// ROWS rows of 32 consecutive slots per warp: tile T = NT * ROWS.  Tiles are handed out by a ticket,
// so the blocks advance through the source as one narrow front and the destination lines they share
// meet in L2.
//
// Stable rank inside the tile without any serial section and without any atomic: every warp owns
// ROWS*32 consecutive slots and a private 16-bit counter per bin of the tile's window (a warp holds at
// most 256 particles of a bin).  Per row, match.any groups the lanes with equal keys; the lowest lane of
// a group reads and advances the warp's counter of that bin, the others take counter + (number of lower
// lanes with the same key).  Rows are taken in slot order, so the rank is the particle's position among
// the warp's particles of that bin BY CONSTRUCTION (no assumption about the order in which the hardware
// serves conflicting shared-memory atomics).  A per-bin pass (8 bins per thread, 128-bit shared accesses
// on packed 16-bit pairs) then turns the 8 per-warp counts into per-warp bases, and
//     destination = offsets[k] + prefix over earlier tiles [t][k] + prefix over earlier warps + rank.
// Only x and vx are loaded up front (the push and the key need nothing else); vy and vz are fetched
// after the ranks are known, so their latency overlaps the per-bin pass and fewer registers are live.
//
// STAGE (electrons): when the tile's particles spread over many bins (runs shorter than 64 slots:
// particles move many cells per step, Eq. 5 violated), the per-bin pass also scans the bin totals,
// the particles are first placed in tile-sorted order in shared memory and then copied out by
// consecutive threads, so that a warp's store covers a few runs instead of 32 separate sectors.
// Windows wider than WA bins are ranked WA bins at a time (direct scatter).
//
// MCCK != 0: the null-collision MCC of the species is folded in (mcc_lane, pic1d_mcc.cuh): the
// destination slot is the particle id, and the velocities are at hand -- in registers on the direct
// path, in the staging buffer on the staged path.
template <int BC, int ROWS, bool STAGE, int MCCK>
__global__ void __launch_bounds__(PIC1D_NT, (STAGE ? 3 : (ROWS <= 4 ? 6 : 4))) k_push_scatter(SortArgs a) {
    extern __shared__ unsigned s_mem[];
    __shared__ int s_tile;
    __shared__ int s_n[2];           // MCCK: candidates, real collisions of the tile
    __shared__ unsigned s_scan[PIC1D_NWARP + 1];
    const int WA = a.WA;             // a multiple of 8
    constexpr int T = PIC1D_NT * ROWS;
    unsigned* s_base = s_mem;        // [WA] absolute destination of the tile's first particle per bin
    unsigned short* s_cnt = reinterpret_cast<unsigned short*>(s_mem + WA);  // [8][WA] per-warp counters, then bases
    const int cnt_words = (STAGE && MCCK) ? max(4 * WA, T / 2) : 4 * WA;      // (the MCC list needs T shorts)
    float* s_st = reinterpret_cast<float*>(s_mem + WA + cnt_words);           // STAGE: [4][T]
    unsigned short* s_key = reinterpret_cast<unsigned short*>(s_st + 4 * T);  // STAGE: [T]
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    unsigned short* my = s_cnt + wp * WA;
    DevSpecies& sp = a.st->sp[a.s];
    const int n_tiles = sp.n_tiles, n_src = sp.n_src, n_push = sp.n_push;
    const uint32_t step = a.st->step;
    int n_refl = 0;  // (counted by the counting pass)
    MccCount mc = {0u, 0u, 0u};
    for (int i = tid; i < cnt_words; i += PIC1D_NT) reinterpret_cast<unsigned*>(s_cnt)[i] = 0u;  // counters are zero between tiles
    if (tid == 0) s_tile = atomicAdd(&sp.ticket2, 1);
    __syncthreads();
    while (true) {
        const int tile = s_tile;
        if (tile >= n_tiles) break;
        const int lo = a.tile_lo[tile], w = a.tile_w[tile], off = a.tile_off[tile];
        const int base = tile * T + wp * (ROWS * 32) + lane;
        const bool full = tile * T + T <= n_push;  // block-uniform
        const int wtot = off < 0 ? 0 : w;          // off < 0: count pool exhausted (sticky error), the tile is lost
        float x[ROWS], vx[ROWS], vy[ROWS], vz[ROWS];
        int rel[ROWS];  // bin relative to the window; -1 = no particle / done
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
        // absolute base of the tile per bin of the first sub-window: in flight together with the particles
        for (int i = tid; i < min(WA, wtot); i += PIC1D_NT)
            s_base[i] = (unsigned)(a.offsets[lo + i] + __ldcg(a.pool + off + i));
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
            const int i = base + r * 32;
            rel[r] = -1;
            if (full || i < n_src) {
                const int key = push_particle<BC>(x[r], vx[r], full || i < n_push, a.E32, a.kappa, a.Nc, a.fNc, a.inv_r, a.shift, a.rp, step, (unsigned)i, n_refl);
                rel[r] = key >= 0 ? key - lo : -1;
            }
        }
        const bool staged = STAGE && wtot <= WA && wtot >= T / 64;  // block-uniform
        for (int sub = 0; sub < wtot; sub += WA) {
            const int nsub = min(WA, wtot - sub);
            // ---- rank inside the warp's segment: match.any groups, the group's lowest lane advances the counter
            unsigned ranked = 0;
#pragma unroll
            for (int r = 0; r < ROWS; ++r) {
                const int k = rel[r] - sub;
                const bool in = rel[r] >= 0 && k < nsub;  // rel < sub only for particles already scattered (-1)
                const unsigned peers = __match_any_sync(0xffffffffu, in ? k : (0x40000000 | lane));
                const int leader = __ffs(peers) - 1;
                unsigned old = 0;
                if (in && lane == leader) { old = my[k]; my[k] = (unsigned short)(old + __popc(peers)); }
                old = __shfl_sync(0xffffffffu, old, leader);
                if (in) {
                    rel[r] = k | ((int)(old + __popc(peers & lanemask_lt())) << 16);
                    ranked |= 1u << r;
                }
                __syncwarp();  // the next row's leaders see the advanced counters
            }
            if (sub == 0) {  // payload: needed only for the stores
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
            }
            __syncthreads();
            // ---- per bin: counts of the 8 warps -> prefix over earlier warps (16-bit pairs packed in 32-bit words)
            // direct: s_cnt = prefix over earlier warps; staged: s_cnt = position in the tile-sorted order,
            // and s_base becomes (absolute destination - position of the bin's first particle)
            unsigned n_out = 0;
            for (int c0 = 0; c0 < nsub; c0 += 8 * PIC1D_NT) {  // 2048 bins per round, in bin order
                const int i8 = c0 + tid * 8;
                const bool act = i8 < nsub;
                uint4 tot = make_uint4(0u, 0u, 0u, 0u);
                if (act) {
#pragma unroll
                    for (int q = 0; q < PIC1D_NWARP; ++q) {
                        const uint4 c = *reinterpret_cast<const uint4*>(s_cnt + q * WA + i8);
                        tot.x += c.x; tot.y += c.y; tot.z += c.z; tot.w += c.w;
                    }
                }
                uint4 b4 = make_uint4(0u, 0u, 0u, 0u);  // packed start per bin
                if (staged) {  // block-wide exclusive scan of the bin totals
                    const unsigned t0 = tot.x & 0xffffu, t1 = tot.x >> 16, t2 = tot.y & 0xffffu, t3 = tot.y >> 16,
                                   t4 = tot.z & 0xffffu, t5 = tot.z >> 16, t6 = tot.w & 0xffffu, t7 = tot.w >> 16;
                    const unsigned S = t0 + t1 + t2 + t3 + t4 + t5 + t6 + t7;
                    unsigned inc = S;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
                        if (lane >= o) inc += t;
                    }
                    if (c0 > 0) __syncthreads();  // s_scan of the previous round has been read
                    if (lane == 31) s_scan[wp] = inc;
                    __syncthreads();
                    unsigned before = 0, all = 0;
#pragma unroll
                    for (int q = 0; q < PIC1D_NWARP; ++q) { const unsigned v = s_scan[q]; if (q < wp) before += v; all += v; }
                    const unsigned e0 = n_out + before + inc - S;
                    n_out += all;
                    const unsigned e1 = e0 + t0, e2 = e1 + t1, e3 = e2 + t2, e4 = e3 + t3, e5 = e4 + t4, e6 = e5 + t5, e7 = e6 + t6;
                    if (act) {
                        uint4 lo4 = *reinterpret_cast<const uint4*>(s_base + i8);
                        uint4 hi4 = *reinterpret_cast<const uint4*>(s_base + i8 + 4);
                        lo4.x -= e0; lo4.y -= e1; lo4.z -= e2; lo4.w -= e3;
                        hi4.x -= e4; hi4.y -= e5; hi4.z -= e6; hi4.w -= e7;
                        *reinterpret_cast<uint4*>(s_base + i8) = lo4;
                        *reinterpret_cast<uint4*>(s_base + i8 + 4) = hi4;
                    }
                    b4 = make_uint4(e0 | (e1 << 16), e2 | (e3 << 16), e4 | (e5 << 16), e6 | (e7 << 16));
                }
                if (act) {
#pragma unroll
                    for (int q = 0; q < PIC1D_NWARP; ++q) {  // counts are re-read: keeping them would spill
                        const uint4 c = *reinterpret_cast<const uint4*>(s_cnt + q * WA + i8);
                        *reinterpret_cast<uint4*>(s_cnt + q * WA + i8) = b4;
                        b4.x += c.x; b4.y += c.y; b4.z += c.z; b4.w += c.w;
                    }
                }
            }
            __syncthreads();
            if (!staged) {
                // ---- direct scatter: destination = tile's base of the bin + prefix over earlier warps + rank
#pragma unroll
                for (int r = 0; r < ROWS; ++r) {
                    const bool act = (ranked >> r) & 1u;
                    const int k = rel[r] & 0xffff;
                    unsigned d = 0;
                    if (act) d = s_base[k] + (unsigned)my[k] + (unsigned)(rel[r] >> 16);
                    if (MCCK) {
                        const int e = mcc_lane<MCCK>(a.m, step, d, act && mcc_null_bit(a.m, d), vx[r], vy[r], vz[r], mc);
                        if (a.m.mask && act) a.m.mask[d] = (uint8_t)e;
                    }
                    if (act) {
                        a.dx[d] = x[r]; a.dvx[d] = vx[r]; a.dvy[d] = vy[r]; a.dvz[d] = vz[r];
                        rel[r] = -1;
                    }
                }
            } else {
                // ---- staged: tile-sorted order in shared memory, then coalesced copy-out ----------------
#pragma unroll
                for (int r = 0; r < ROWS; ++r) {
                    if (!((ranked >> r) & 1u)) continue;
                    const int k = rel[r] & 0xffff;
                    const unsigned li = (unsigned)my[k] + (unsigned)(rel[r] >> 16);
                    s_st[li] = x[r]; s_st[T + li] = vx[r]; s_st[2 * T + li] = vy[r]; s_st[3 * T + li] = vz[r];
                    s_key[li] = (unsigned short)k;
                    rel[r] = -1;
                }
                if (MCCK && tid == 0) s_n[1] = 0;
                __syncthreads();
                if (!MCCK) {
                    for (int j = tid; j < (int)n_out; j += PIC1D_NT) {
                        const unsigned d = s_base[s_key[j]] + (unsigned)j;
                        a.dx[d] = s_st[j]; a.dvx[d] = s_st[T + j]; a.dvy[d] = s_st[2 * T + j]; a.dvz[d] = s_st[3 * T + j];
                    }
                } else {
                    // The collisions, folded in: the destination slot is the particle id, the velocities are in
                    // the staging buffer.  Copy-out and null-test look-ups of the whole tile first (all in flight
                    // together), then the process selection of the candidates, row by row; the real collisions go
                    // to a list (the per-warp counters are free by now and hold it) ...
                    unsigned short* s_rl = s_cnt;  // [T] real collisions: j | event << 12
                    unsigned dj[ROWS], nw[ROWS];
#pragma unroll
                    for (int it = 0; it < ROWS; ++it) {
                        const int j = it * PIC1D_NT + tid;
                        dj[it] = 0u; nw[it] = 0u;
                        if (j < (int)n_out) {
                            const unsigned d = s_base[s_key[j]] + (unsigned)j;
                            dj[it] = d;
                            nw[it] = __ldcg(a.m.null_bits + (d >> 5));
                            a.dx[d] = s_st[j]; a.dvx[d] = s_st[T + j]; a.dvy[d] = s_st[2 * T + j]; a.dvz[d] = s_st[3 * T + j];
                            if (a.m.mask) a.m.mask[d] = 0;
                        }
                    }
#pragma unroll
                    for (int it = 0; it < ROWS; ++it) {
                        const int j = it * PIC1D_NT + tid;
                        const unsigned d = dj[it];
                        const bool cand = j < (int)n_out && ((nw[it] >> (d & 31u)) & 1u);
                        if (!__any_sync(0xffffffffu, cand)) continue;
                        uint32_t b0[4];
                        const int e = mcc_event<MCCK>(a.m, step, d, cand, s_st[T + j], s_st[2 * T + j], s_st[3 * T + j], mc, b0);
                        if (a.m.mask && e) a.m.mask[d] = (uint8_t)e;
                        const int idx = warp_append(e != 0, &s_n[1]);
                        if (e) s_rl[idx] = (unsigned short)(j | (e << 12));
                    }
                    __syncthreads();
                    // ... and get their kinematics one thread per real collision
                    const int n_coll = s_n[1];
                    for (int c = tid; c < n_coll; c += PIC1D_NT) {  // one thread per real collision: kinematics
                        const int j = s_rl[c] & 0xfff, e = s_rl[c] >> 12;
                        const unsigned d = s_base[s_key[j]] + (unsigned)j;
                        uint32_t b0[4];
                        philox4x32_10(d, step, STREAM_COLL + (uint32_t)a.m.s, 0u, a.m.k0, a.m.k1, b0);
                        float cx = s_st[T + j], cy = s_st[2 * T + j], cz = s_st[3 * T + j];
                        mcc_kinematics<MCCK>(a.m, step, d, e, b0, cx, cy, cz);
                        a.dvx[d] = cx; a.dvy[d] = cy; a.dvz[d] = cz;  // overwrites the copy-out of this block
                    }
                }
            }
            __syncthreads();
            // ---- zero the counters again; next sub-window's bases ---------------------------------------
            {
                if (MCCK && staged) {  // the collision list lay over the counters
                    for (int i8 = tid * 8; i8 < T; i8 += 8 * PIC1D_NT)
                        *reinterpret_cast<uint4*>(s_cnt + i8) = make_uint4(0u, 0u, 0u, 0u);
                }
                for (int i8 = tid * 8; i8 < nsub; i8 += 8 * PIC1D_NT) {
#pragma unroll
                    for (int q = 0; q < PIC1D_NWARP; ++q)
                        *reinterpret_cast<uint4*>(s_cnt + q * WA + i8) = make_uint4(0u, 0u, 0u, 0u);
                }
                for (int i = tid; i < nsub; i += PIC1D_NT) {
                    const int kk = sub + WA + i;
                    if (kk < wtot) s_base[i] = (unsigned)(a.offsets[lo + kk] + __ldcg(a.pool + off + kk));
                }
            }
            if (sub + WA < wtot) __syncthreads();
        }
        if (tid == 0) s_tile = atomicAdd(&sp.ticket2, 1);
        __syncthreads();
    }
    if (MCCK) mcc_flush_counts(a.m, mc);
}

// ---- set up the sorts of one step ------------------------------------------------------------------
// mode 0: initial sort after a load (nothing is pushed); mode 1: a regular step, which also advances the
// device-resident step index (every kernel reads the step from DevState, never from a host argument, so
// a captured CUDA graph of the step can be replayed).
struct BeginArgs {
    DevState* st;
    int n_species, mode;
    int T[2];
    int *grp_lo[2], *grp_hi[2];
    int n_groups[2];
    int* ion_nb;   // per-MCC-tile ionisation counts of the electron set (may be null)
    int n_ion_nb;
};

__global__ void k_step_begin(BeginArgs b) {
    DevState* st = b.st;
    const int tid = threadIdx.x + blockIdx.x * blockDim.x, nthr = blockDim.x * gridDim.x;
    if (tid == 0) {
        for (int s = 0; s < b.n_species; ++s) {
            DevSpecies& sp = st->sp[s];
            sp.n_push = b.mode ? sp.n_live : 0;
            sp.n_src = sp.n_live;
            sp.n_tiles = (sp.n_live + b.T[s] - 1) / b.T[s];
            sp.n_dead = 0;
            sp.pool_used = 0;
            sp.ticket = 0;
            sp.ticket2 = 0;
            sp.scan_done = 0;
            sp.dead_done = 0;
        }
        st->n_abs = 0;
        if (b.mode) { st->step = st->step_next; st->step_next = st->step + 1u; }
    }
    for (int s = 0; s < b.n_species; ++s)
        for (int i = tid; i < b.n_groups[s]; i += nthr) { b.grp_lo[s][i] = 0x7fffffff; b.grp_hi[s][i] = -1; }
    for (int i = tid; i < b.n_ion_nb; i += nthr) b.ion_nb[i] = 0;
}

// ---- secondary-electron emission at ion impact (L41; R19) --------------------------------
struct SeeArgs {
    DevState* st;
    const unsigned* abs_list;
    int abs_cap;
    float *ex, *evx, *evy, *evz;  // electron SOURCE buffer of this step (injected after the survivors)
    int cap_e;
    int T;
    float gamma, vth, fNc;
    uint32_t k0, k1;
};

__global__ void __launch_bounds__(1024) k_see_emit(SeeArgs a) {
    __shared__ int s_w[32];
    __shared__ int s_run, s_tot;
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    DevState* st = a.st;
    int n_abs = st->sp[1].n_dead;
    if (n_abs > a.abs_cap) {
        n_abs = a.abs_cap;
        if (tid == 0) atomicOr(&st->err, ERRBIT_CAPACITY);
    }
    const int ne = st->sp[0].n_live;
    const uint32_t step = st->step;
    if (tid == 0) s_run = 0;
    __syncthreads();
    for (int base = 0; base < n_abs; base += 1024) {
        const int i = base + tid;
        bool emit = false;
        uint32_t w[4];
        unsigned slot = 0, wall = 0;
        if (i < n_abs) {
            const unsigned e = a.abs_list[i];
            slot = e & 0x7fffffffu; wall = e >> 31;
            philox4x32_10(slot, step, STREAM_SEE, 0u, a.k0, a.k1, w);
            emit = u01(w[0]) < a.gamma;
        }
        const unsigned bal = __ballot_sync(0xffffffffu, emit);
        if (lane == 0) s_w[wp] = __popc(bal);
        __syncthreads();
        if (wp == 0) {  // exclusive prefix over the 32 warps, chunk total
            const int t = s_w[lane];
            int ti = t;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int u = __shfl_up_sync(0xffffffffu, ti, o);
                if (lane >= o) ti += u;
            }
            s_w[lane] = ti - t;
            if (lane == 31) s_tot = ti;
        }
        __syncthreads();
        const int idx = s_run + s_w[wp] + __popc(bal & lanemask_lt());  // ascending ion-slot order
        if (emit) {
            const int d = ne + idx;
            if (d < a.cap_e) {
                uint32_t w2[4];
                philox4x32_10(slot, step, STREAM_SEE, 1u, a.k0, a.k1, w2);
                const float u1 = u01(w[1]), u2 = u01(w[2]), u3 = u01(w[3]), u4 = u01(w2[0]);
                float x, sgn;
                if (wall == 0) { x = u1; sgn = 1.0f; }
                else { x = fminf(__fsub_rn(a.fNc, __fsub_rn(1.0f, u1)), nextafterf(a.fNc, 0.0f)); sgn = -1.0f; }
                const float rx = sqrtf(__fmul_rn(-2.0f, logf(__fsub_rn(1.0f, u2))));
                const float rt = sqrtf(__fmul_rn(-2.0f, logf(__fsub_rn(1.0f, u3))));
                const float ph = __fmul_rn(6.2831855f, u4);
                a.ex[d] = x;
                a.evx[d] = __fmul_rn(sgn, __fmul_rn(a.vth, rx));
                a.evy[d] = __fmul_rn(a.vth, __fmul_rn(rt, cosf(ph)));
                a.evz[d] = __fmul_rn(a.vth, __fmul_rn(rt, sinf(ph)));
            }
        }
        __syncthreads();
        if (tid == 0) s_run += s_tot;
        __syncthreads();
    }
    if (tid == 0) {
        const int emitted = s_run;
        const int room = a.cap_e - ne;
        const int kept = emitted < room ? emitted : (room > 0 ? room : 0);
        DevSpecies& se = st->sp[0];
        se.n_src = ne + kept;
        se.n_tiles = (se.n_src + a.T - 1) / a.T;
        se.injected += (ull)kept;
        if (emitted > kept) { se.dropped += (ull)(emitted - kept); atomicOr(&st->err, ERRBIT_CAPACITY); }
        st->n_abs = n_abs;
    }
}
