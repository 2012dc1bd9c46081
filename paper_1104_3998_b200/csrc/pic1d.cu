// pic1d.cu -- C-ABI (include/pic1d.h) and step orchestration of the B200-native PIC/MCC hot path.
//
// One stream-ordered kernel sequence per step, no host round trip (contrast PAPER.md L144):
//   k_step_begin
//   per species (ions first, so their wall hits can emit secondaries into the electron source):
//       k_push_count[_w] -> k_bin_scan (prefix over tiles per sort cell + the offsets scan, last block done)
//       -> k_push_scatter[_w] (species with sparse candidates: MCC folded in) [-> k_see_emit after the ions]
//       (_w: barrier-free warp-tile kernels for species that obey Eq. 5, pic1d_sort_warp.cuh)
//   main stream: k_deposit (one launch, every species) -> k_field[_smem] (rho combine + Poisson + E)
//   side stream, beside them: k_mcc -> k_mcc_births per species with a pass of its own, k_null_bits_next (the
//       null-test masks of the folded species for the NEXT step), [k_coulomb]
// 13 launches for config 4; pairs of steps are replayed from a captured CUDA graph (pic1d_step).
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -fmad=false (see ../build.py).
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/pic1d.h"
#include "pic1d_device.cuh"
#include "pic1d_mcc.cuh"
#include "pic1d_sort.cuh"
#include "pic1d_sort_warp.cuh"
#include "pic1d_grid.cuh"
#include "pic1d_coulomb.cuh"

namespace {

struct SpeciesHost {
    float* buf[2][4];
    int cur;
    int capacity, n_tiles_max, n_groups_max;
    int T;            // slots per sort tile: 2048 / 1024 (block tiles) or PIC1D_TW (warp tiles)
    bool warp_tiles;  // the species obeys Eq. 5: barrier-free warp-tile kernels (pic1d_sort_warp.cuh)
    int *tile_lo, *tile_w, *tile_off, *tile_dead, *grp_lo, *grp_hi, *pool;
    int pool_size, pool_stride, pool_fixed;
    int *hist, *offsets, *keys_dbg, *partner;
    uint8_t* mask;
    double *part, *side, *rho_s;
    int n_mcc_tiles;
    unsigned* null_bits;  // folded MCC: null-test bit per sorted slot of this step
    int mcck;  // 0: the MCC of the species is a pass of its own (k_mcc) or absent; 1 / 2: folded into the scatter
};

struct TimeMark {
    const char* name;
    int species;
    cudaEvent_t ev;
};

}  // namespace

struct pic1d {
    pic1d_config_t cfg;
    cudaStream_t stream;
    int nodes, n_sc, T, G, n_dep_blocks, num_sms;
    float inv_r;
    SpeciesHost sp[2];
    DevState* st;
    double *rho, *phi, *E, *S, *Tt, *mom_partial;
    float* E32;
    unsigned* abs_list;
    int abs_cap;
    unsigned* ion_bits;  // ionisation records of the electron set (pic1d_mcc.cuh)
    float* ion_gp;
    int* ion_nb;
    int n_ion_words;
    ull* eedf_dev;
    int eedf_cap;
    uint32_t step;
    int loaded_mask;
    bool ready;
    int64_t launches;
    cudaError_t last_err;
    int grid_count[2], grid_scatter[2][2], WA;
    size_t smem_sort, smem_count[2], smem_scatter[2];
    void (*k_count[2])(SortArgs);
    void (*k_scatter[2][2])(SortArgs);  // [species][0 plain | 1 the step's, with the MCC folded in]
    cudaStream_t side;              // collisions run here beside the deposit and the field solve
    cudaEvent_t ev_fork, ev_join;
    bool null_ready;                // the null-test masks of the NEXT step have been enqueued (by the previous step)
    cudaGraphExec_t graph[4];       // two captured steps, per parity of BOTH species' sort buffers at their start
    bool graph_off;                 // a capture or an instantiation failed once: plain launches from then on
    int64_t graph_launches;         // replays so far
    int64_t launches_per_2steps;
    bool timing;
    std::vector<TimeMark> marks;
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used;
};

namespace {

const int MOM_BLOCKS = 1024;
const double PIC1D_FOLD_P0_MAX = 0.25;
const int EEDF_MAX_BINS = 65536;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

template <class Tp>
Tp* carve(char* base, size_t& off, size_t count) {
    off = align_up(off, 256);
    Tp* p = base ? reinterpret_cast<Tp*>(base + off) : nullptr;
    off += count * sizeof(Tp);
    return p;
}

int pow2_floor(int v) {
    int p = 1;
    while (p * 2 <= v) p *= 2;
    return p;
}

int validate_cfg(const pic1d_config_t* c) {
    if (!c || c->struct_size != sizeof(pic1d_config_t)) return PIC1D_ERR_ARG;
    if (c->n_cells < 2 || c->n_cells > (1 << 24)) return PIC1D_ERR_ARG;
    if (c->bc != 0 && c->bc != 1) return PIC1D_ERR_ARG;
    if (c->n_species < 1 || c->n_species > PIC1D_MAX_SPECIES) return PIC1D_ERR_ARG;
    if (!(c->sort_inv_ratio > 0.0)) return PIC1D_ERR_ARG;
    int e;
    double m = std::frexp(c->sort_inv_ratio, &e);
    if (m != 0.5) return PIC1D_ERR_ARG;  // power of two: x * inv_r is exact (R9)
    double nsc = std::ceil((double)c->n_cells * c->sort_inv_ratio);
    if (nsc < 1 || nsc > 49152) return PIC1D_ERR_ARG;  // one int counter per sort cell in shared memory
    for (int s = 0; s < c->n_species; ++s) {
        int64_t cap = c->sp[s].capacity;
        if (cap < 4096 || cap % 4096 != 0 || cap > (1ll << 30)) return PIC1D_ERR_ARG;
        if (!(c->coul_A[s] >= 0.0) || !std::isfinite(c->coul_A[s])) return PIC1D_ERR_ARG;  // 0 = off
    }
    if (!(c->e_reflect >= 0.0 && c->e_reflect <= 1.0)) return PIC1D_ERR_ARG;  // a probability (also rejects NaN)
    return PIC1D_OK;
}

// Lay the handle's device arrays out in the caller's workspace (base == nullptr: size query only).
size_t layout(pic1d* h, char* base) {
    const pic1d_config_t& c = h->cfg;
    h->nodes = c.bc == 1 ? c.n_cells : c.n_cells + 1;
    h->n_sc = (int)std::ceil((double)c.n_cells * c.sort_inv_ratio);
    h->inv_r = (float)c.sort_inv_ratio;
    int64_t cap_max = 0;
    for (int s = 0; s < c.n_species; ++s) cap_max = std::max<int64_t>(cap_max, c.sp[s].capacity);
    h->T = cap_max >= 2048ll * 592 ? 2048 : 1024;
    const int rr = c.sort_inv_ratio < 1.0 ? (int)std::llround(1.0 / c.sort_inv_ratio) : 1;
    const int ppc_est = (int)std::max<int64_t>(1, cap_max / c.n_cells);
    // cells per deposit block: ~32-64 k particles per block, but at least ~300 blocks when the grid allows
    const int g_work = pow2_floor(std::max(1, 65536 / ppc_est)), g_par = pow2_floor(std::max(1, c.n_cells / 296));
    h->G = std::min(2048, std::max(rr, std::min(g_work, g_par)));
    h->n_dep_blocks = (c.n_cells + h->G - 1) / h->G;
    size_t off = 0;
    h->st = carve<DevState>(base, off, 1);
    h->rho = carve<double>(base, off, h->nodes + 1);
    h->phi = carve<double>(base, off, h->nodes + 1);
    h->E = carve<double>(base, off, h->nodes + 1);
    h->S = carve<double>(base, off, h->nodes + 1);
    h->Tt = carve<double>(base, off, h->nodes + 1);
    h->E32 = carve<float>(base, off, h->nodes + 1);
    h->mom_partial = carve<double>(base, off, MOM_BLOCKS * 5);
    h->eedf_cap = EEDF_MAX_BINS;
    h->eedf_dev = carve<ull>(base, off, EEDF_MAX_BINS);
    h->abs_cap = 0;
    h->abs_list = nullptr;
    if (c.n_species > 1 && c.see_gamma > 0.0 && c.bc == 0) {
        h->abs_cap = (int)std::min<int64_t>(c.sp[1].capacity, std::max<int64_t>(1 << 20, c.sp[1].capacity / 16));
        h->abs_list = carve<unsigned>(base, off, h->abs_cap);
    }
    for (int s = 0; s < c.n_species; ++s) {
        SpeciesHost& p = h->sp[s];
        p.capacity = (int)c.sp[s].capacity;
        p.cur = 0;
        for (int b = 0; b < 2; ++b)
            for (int k = 0; k < 4; ++k) p.buf[b][k] = carve<float>(base, off, p.capacity);
        // ions always; electrons only on the caller's word: they may move many cells per step (configs 2-4)
        p.warp_tiles = s != 0 || (c.flags & PIC1D_FLAG_EQ5_ELECTRONS) != 0;
        p.T = p.warp_tiles ? PIC1D_TW : h->T;
        p.n_tiles_max = p.capacity / p.T;
        p.n_groups_max = (p.n_tiles_max + PIC1D_GROUP - 1) / PIC1D_GROUP;
        p.tile_lo = carve<int>(base, off, p.n_tiles_max);
        p.tile_w = carve<int>(base, off, p.n_tiles_max);
        p.tile_off = carve<int>(base, off, p.n_tiles_max);
        p.tile_dead = carve<int>(base, off, p.n_tiles_max);
        p.grp_lo = carve<int>(base, off, p.n_groups_max);
        p.grp_hi = carve<int>(base, off, p.n_groups_max);
        // count pool: one fixed row of pool_stride bins per tile + an overflow region for wider windows
        const int64_t over = std::max<int64_t>(4 << 20, p.capacity);  // see pic1d.h, "Displacement limits"
        int64_t stride = p.warp_tiles ? PIC1D_PSW : std::min<int64_t>((h->n_sc + 3) / 4 * 4, 4096);
        if (!p.warp_tiles) stride = std::max<int64_t>(4, std::min<int64_t>(stride, (((1ll << 31) - 1 - over) / p.n_tiles_max) / 4 * 4));
        p.pool_stride = (int)stride;
        p.pool_fixed = (int)(stride * p.n_tiles_max);
        p.pool_size = (int)(p.pool_fixed + over);
        p.pool = carve<int>(base, off, p.pool_size);
        p.hist = carve<int>(base, off, h->n_sc + 1);
        p.offsets = carve<int>(base, off, h->n_sc + 1);
        p.keys_dbg = nullptr;
        p.mask = nullptr;
        p.partner = nullptr;
        if (c.flags & PIC1D_FLAG_CAPTURE) {
            p.keys_dbg = carve<int>(base, off, p.capacity);
            p.mask = carve<uint8_t>(base, off, p.capacity);
            if (c.coul_A[s] > 0.0) p.partner = carve<int>(base, off, p.capacity);
        }
        p.part = carve<double>(base, off, (size_t)h->n_dep_blocks * h->G);
        p.side = carve<double>(base, off, h->n_dep_blocks);
        p.rho_s = carve<double>(base, off, h->nodes + 1);
        p.n_mcc_tiles = (p.capacity + MCC_TILE - 1) / MCC_TILE;
        // fold the species' MCC into its scatter when its null-test candidates are sparse (the scatter's idle
        // issue slots absorb them); a species most of whose particles are candidates keeps the compacting
        // pass of its own (k_mcc) -- measured, DESIGN.md section 6.  The flags force either choice.
        const bool sparse = c.sp[s].P0 <= PIC1D_FOLD_P0_MAX;
        p.mcck = (c.flags & PIC1D_FLAG_NO_FOLD) ? 0 : (((c.flags & PIC1D_FLAG_FOLD_ALL) || sparse) ? c.sp[s].mcc_kind : 0);
        p.null_bits = p.mcck ? carve<unsigned>(base, off, p.capacity / 32) : nullptr;
    }
    h->ion_bits = nullptr; h->ion_gp = nullptr; h->ion_nb = nullptr; h->n_ion_words = 0;
    if (c.sp[0].mcc_kind == 1) {
        h->n_ion_words = h->sp[0].capacity / 32;
        h->ion_bits = carve<unsigned>(base, off, h->n_ion_words);
        h->ion_gp = carve<float>(base, off, h->sp[0].capacity);
        h->ion_nb = carve<int>(base, off, h->sp[0].n_mcc_tiles);
    }
    return align_up(off, 256);
}

bool ck(pic1d* h, cudaError_t e) {
    if (e != cudaSuccess) { h->last_err = e; return false; }
    return true;
}

void mark(pic1d* h, const char* name, int species) {
    h->launches++;
    if (!h->timing) return;
    if (h->ev_used == h->ev_pool.size()) {
        cudaEvent_t e;
        cudaEventCreate(&e);
        h->ev_pool.push_back(e);
    }
    cudaEvent_t e = h->ev_pool[h->ev_used++];
    cudaEventRecord(e, h->stream);
    h->marks.push_back(TimeMark{name, species, e});
}

MccP mcc_params(pic1d* h, int s) {
    const pic1d_config_t& c = h->cfg;
    MccP m;
    memset(&m, 0, sizeof(m));
    m.st = h->st; m.mask = h->sp[s].mask; m.null_bits = h->sp[s].null_bits;
    m.ion_bits = h->ion_bits; m.ion_gp = h->ion_gp; m.ion_nb = h->ion_nb;
    m.s = s; m.kind = c.sp[s].mcc_kind;
    m.k0 = (uint32_t)c.seed; m.k1 = (uint32_t)(c.seed >> 32);
    m.inv_g_cap = (float)c.sp[s].inv_g_cap; m.c_eV = (float)c.sp[s].c_eV;
    m.r_el = (float)c.r_el; m.r_exc = (float)c.r_exc; m.r_ion = (float)c.r_ion;
    m.E_exc = (float)c.E_exc; m.E_ion = (float)c.E_ion;
    m.two_mr = (float)(2.0 * c.mass_ratio); m.gvt = (float)c.gas_vth_ion;
    // null test in integers: U(w) = (w >> 8) 2^-24 < P0  <=>  (w >> 8) < ceil(P0 2^24)  <=>  w <= null_le
    const uint64_t thr = (uint64_t)std::ceil((double)(float)c.sp[s].P0 * 16777216.0) << 8;
    m.null_any = thr > 0;
    m.null_le = (uint32_t)(thr - 1);
    return m;
}

SortArgs sort_args(pic1d* h, int s) {
    SpeciesHost& p = h->sp[s];
    SortArgs a;
    const int c = p.cur, d = c ^ 1;
    a.sx = p.buf[c][0]; a.svx = p.buf[c][1]; a.svy = p.buf[c][2]; a.svz = p.buf[c][3];
    a.dx = p.buf[d][0]; a.dvx = p.buf[d][1]; a.dvy = p.buf[d][2]; a.dvz = p.buf[d][3];
    a.E32 = h->E32; a.st = h->st; a.s = s;
    a.tile_lo = p.tile_lo; a.tile_w = p.tile_w; a.tile_off = p.tile_off; a.tile_dead = p.tile_dead;
    a.grp_lo = p.grp_lo; a.grp_hi = p.grp_hi; a.pool = p.pool; a.pool_size = p.pool_size; a.pool_stride = p.pool_stride; a.pool_fixed = p.pool_fixed;
    a.hist = p.hist; a.offsets = p.offsets; a.keys_dbg = p.keys_dbg;
    a.abs_list = (s == 1) ? h->abs_list : nullptr;
    a.abs_cap = h->abs_cap;
    a.kappa = (float)h->cfg.sp[s].kappa;
    a.fNc = (float)h->cfg.n_cells; a.inv_r = h->inv_r; a.Nc = h->cfg.n_cells; a.n_sc = h->n_sc;
    a.shift = 0; a.WA = h->WA;
    a.m = mcc_params(h, s);
    a.rp.prob = (s == 0 && h->cfg.bc == 0) ? (float)h->cfg.e_reflect : 0.0f;
    a.rp.k0 = (uint32_t)h->cfg.seed; a.rp.k1 = (uint32_t)(h->cfg.seed >> 32);
    return a;
}

typedef void (*sort_kernel_t)(SortArgs);

sort_kernel_t count_kernel(int bc, int T) {
    if (bc == 1) return T == 2048 ? k_push_count<1, 2> : k_push_count<1, 1>;
    return T == 2048 ? k_push_count<0, 2> : k_push_count<0, 1>;
}

// block tiles (species 0 only).  stage: the species may spread a tile over many bins (electrons), see
// k_push_scatter; mcck: the electron collision set is folded in
template <int BC, int MCCK>
sort_kernel_t scatter_kernel_bm(int T, bool stage) {
    if (stage) return T == 2048 ? k_push_scatter<BC, 8, true, MCCK> : k_push_scatter<BC, 4, true, MCCK>;
    return T == 2048 ? k_push_scatter<BC, 8, false, MCCK> : k_push_scatter<BC, 4, false, MCCK>;
}
sort_kernel_t scatter_kernel(int bc, int T, bool stage, int mcck) {
    if (bc == 1) return mcck == 1 ? scatter_kernel_bm<1, 1>(T, stage) : scatter_kernel_bm<1, 0>(T, stage);
    return mcck == 1 ? scatter_kernel_bm<0, 1>(T, stage) : scatter_kernel_bm<0, 0>(T, stage);
}

// warp tiles.  abs: the species records its absorbed slots (ions with secondary emission)
template <int BC, bool ABS>
sort_kernel_t scatter_kernel_wm(int mcck) {
    if (mcck == 1) return k_push_scatter_w<BC, ABS, 1>;
    if (mcck == 2) return k_push_scatter_w<BC, ABS, 2>;
    return k_push_scatter_w<BC, ABS, 0>;
}
sort_kernel_t scatter_kernel_w(int bc, bool abs, int mcck) {
    if (bc == 1) return scatter_kernel_wm<1, false>(mcck);
    return abs ? scatter_kernel_wm<0, true>(mcck) : scatter_kernel_wm<0, false>(mcck);
}

int occupancy_grid(pic1d* h, sort_kernel_t kernel, size_t smem) {
    if (smem > 48 * 1024) cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int nb = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, PIC1D_NT, smem);
    return std::max(1, nb) * h->num_sms;
}

// per species two scatter kernels: [0] plain (the passes of a load sort nothing but particles), [1] the
// step's (with the species' MCC folded in, unless PIC1D_FLAG_NO_FOLD)
void setup_launch(pic1d* h) {
    cudaFuncSetAttribute(k_field_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, FIELD_SMEM_MAX * (int)sizeof(double));
    cudaFuncSetAttribute(k_coulomb, cudaFuncAttributeMaxDynamicSharedMemorySize, 6144 * 12);
    cudaFuncSetAttribute(k_mcc<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(3 * MCC_TILE * sizeof(float)));
    cudaFuncSetAttribute(k_mcc<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(3 * MCC_TILE * sizeof(float)));
    h->WA = std::min((h->n_sc + 1 + 7) / 8 * 8, PIC1D_WA_MAX);
    h->smem_sort = (size_t)(h->WA + 1) * sizeof(int);
    for (int s = 0; s < h->cfg.n_species; ++s) {
        SpeciesHost& p = h->sp[s];
        const bool abs = s == 1 && h->abs_list != nullptr;
        for (int v = 0; v < 2; ++v) {
            const int mcck = v ? p.mcck : 0;
            if (p.warp_tiles) {
                h->k_count[s] = h->cfg.bc == 1 ? k_push_count_w<1> : k_push_count_w<0>;
                h->k_scatter[s][v] = scatter_kernel_w(h->cfg.bc, abs, mcck);
                h->smem_count[s] = 0;
                h->smem_scatter[s] = 0;
            } else {
                const bool stage = s == 0;
                h->k_count[s] = count_kernel(h->cfg.bc, h->T);
                h->k_scatter[s][v] = scatter_kernel(h->cfg.bc, h->T, stage, mcck);
                h->smem_count[s] = h->smem_sort;
                h->smem_scatter[s] = (size_t)h->WA * 4 + (stage ? std::max<size_t>((size_t)h->WA * 16, (size_t)h->T * 2) + (size_t)h->T * 18 : (size_t)h->WA * 16);
            }
            h->grid_scatter[s][v] = occupancy_grid(h, h->k_scatter[s][v], h->smem_scatter[s]);
        }
        h->grid_count[s] = occupancy_grid(h, h->k_count[s], h->smem_count[s]);
    }
}

// fine sort of species s.  in_step: 1 = a regular step (push, folded MCC); 0 = a pass of a load's sort
void enqueue_sort(pic1d* h, int s, int in_step, int shift = 0) {
    SpeciesHost& p = h->sp[s];
    SortArgs a = sort_args(h, s);
    if (shift > 0) {  // coarse pass of an unsorted load: sort by (sort cell >> shift)
        a.shift = shift;
        a.n_sc = ((h->n_sc - 1) >> shift) + 1;
    }
    const int tiles_per_block = p.warp_tiles ? PIC1D_NWARP : 1;
    const int nb_max = (p.n_tiles_max + tiles_per_block - 1) / tiles_per_block;
    const int gc = std::min(h->grid_count[s], nb_max), gs = std::min(h->grid_scatter[s][in_step], nb_max);
    h->k_count[s]<<<gc, PIC1D_NT, h->smem_count[s], h->stream>>>(a);
    mark(h, "push_count", s);
    const bool fold = in_step && p.mcck;
    a.null_first = a.abs_list ? PIC1D_DEAD_CHUNKS : 0;  // blocks that scan the per-tile absorbed counts
    const int nb_bins = (a.n_sc + 31) / 32;
    const int nw = (nb_bins < h->num_sms && p.n_tiles_max >= 4096) ? 32 : 16;  // warps per block (see k_bin_scan)
    const int nb_null = (fold && !h->null_ready) ? (p.capacity / 32 + nw * 32 - 1) / (nw * 32) : 0;
    if (nw == 16) k_bin_scan<16><<<nb_bins + a.null_first + nb_null, 16 * 32, 0, h->stream>>>(a);
    else k_bin_scan<32><<<nb_bins + a.null_first + nb_null, 32 * 32, 0, h->stream>>>(a);
    mark(h, "bin_scan", s);
    h->k_scatter[s][in_step]<<<gs, PIC1D_NT, h->smem_scatter[s], h->stream>>>(a);
    mark(h, "push_scatter", s);
    p.cur ^= 1;
}

void enqueue_begin(pic1d* h, int mode) {
    const int ns = h->cfg.n_species;
    BeginArgs b;
    memset(&b, 0, sizeof(b));
    b.st = h->st; b.n_species = ns; b.mode = mode;
    for (int s = 0; s < ns; ++s) {
        b.T[s] = h->sp[s].T; b.grp_lo[s] = h->sp[s].grp_lo; b.grp_hi[s] = h->sp[s].grp_hi;
        b.n_groups[s] = h->sp[s].n_groups_max;
    }
    b.ion_nb = h->ion_nb; b.n_ion_nb = h->ion_nb ? h->sp[0].n_mcc_tiles : 0;
    k_step_begin<<<4, 256, 0, h->stream>>>(b);
    mark(h, "step_begin", -1);
}

// deposit of every species (one launch) + edge nodes, rho, Poisson and E (one block)
void enqueue_grid(pic1d* h, int in_step) {
    const pic1d_config_t& c = h->cfg;
    DepositArgs d;
    memset(&d, 0, sizeof(d));
    FieldArgs f;
    memset(&f, 0, sizeof(f));
    CombineArgs& cb = f.cb;
    for (int s = 0; s < c.n_species; ++s) {
        SpeciesHost& p = h->sp[s];
        d.sp[s].x = p.buf[p.cur][0]; d.sp[s].offsets = p.offsets; d.sp[s].part = p.part; d.sp[s].side = p.side;
        cb.part[s] = p.part; cb.side[s] = p.side; cb.rho_s[s] = p.rho_s; cb.sign[s] = c.sp[s].charge_sign;
    }
    d.Nc = c.n_cells; d.n_sc = h->n_sc; d.G = h->G; d.inv_r = h->inv_r;
    k_deposit<<<dim3(h->n_dep_blocks, c.n_species), PIC1D_NT, (h->G + 1) * (sizeof(ull) + 3 * sizeof(unsigned)), h->stream>>>(d);
    mark(h, "deposit", -1);
    cb.rho = h->rho; cb.n_species = c.n_species; cb.Nc = c.n_cells; cb.nodes = h->nodes; cb.G = h->G;
    cb.bc = c.bc; cb.background = c.background_rho;
    f.rho = h->rho; f.phi = h->phi; f.E = h->E; f.S = h->S; f.Tt = h->Tt; f.E32 = h->E32;
    f.Nc = c.n_cells; f.nodes = h->nodes; f.bc = c.bc; f.V0 = c.V0_norm; f.omega_dt = c.omega_dt;
    f.st = h->st; f.in_step = in_step;
    if (c.n_cells <= FIELD_SMEM_MAX) {
        const size_t sm = (size_t)((c.n_cells + 1023) / 1024) * 32 * 32 * sizeof(double);
        k_field_smem<<<1, 1024, sm, h->stream>>>(f);
    } else {
        k_field<<<1, 1024, 0, h->stream>>>(f);
    }
    mark(h, "field", -1);
}

MccArgs mcc_args(pic1d* h, int s) {
    const pic1d_config_t& c = h->cfg;
    SpeciesHost& p = h->sp[s];
    SpeciesHost& pe = h->sp[0];
    MccArgs m;
    memset(&m, 0, sizeof(m));
    m.x = p.buf[p.cur][0]; m.vx = p.buf[p.cur][1]; m.vy = p.buf[p.cur][2]; m.vz = p.buf[p.cur][3];
    m.ex = pe.buf[pe.cur][0]; m.evx = pe.buf[pe.cur][1]; m.evy = pe.buf[pe.cur][2]; m.evz = pe.buf[pe.cur][3];
    m.cap_e = pe.capacity;
    if (c.n_species > 1) {
        SpeciesHost& pi = h->sp[1];
        m.ix = pi.buf[pi.cur][0]; m.ivx = pi.buf[pi.cur][1]; m.ivy = pi.buf[pi.cur][2]; m.ivz = pi.buf[pi.cur][3];
        m.cap_i = pi.capacity;
    }
    m.m = mcc_params(h, s);
    m.n_species = c.n_species;
    return m;
}

// the collisions that are not folded into a scatter, and the ionisation pairs.  They depend on the sorted
// particles only (not on rho or E, R3), so in a step they run on the side stream, beside the
// deposit and the field solve.
void enqueue_mcc(pic1d* h, cudaStream_t st) {
    const pic1d_config_t& c = h->cfg;
    for (int s = 0; s < c.n_species; ++s) {
        const int kind = c.sp[s].mcc_kind;
        if (kind == 0) continue;
        SpeciesHost& p = h->sp[s];
        MccArgs m = mcc_args(h, s);
        if (p.mcck == 0) {
            // dense candidates: the tile's velocities are streamed into shared memory by bulk async copies
            const bool stage = c.sp[s].P0 > PIC1D_FOLD_P0_MAX && !(c.flags & PIC1D_FLAG_MCC_GATHER);
            const int grid = std::min(p.n_mcc_tiles, h->num_sms * (stage ? 3 : 4));
            const size_t sm = stage ? 3 * MCC_TILE * sizeof(float) : 0;
            if (kind == 1) { if (stage) k_mcc<1, true><<<grid, PIC1D_NT, sm, st>>>(m); else k_mcc<1, false><<<grid, PIC1D_NT, 0, st>>>(m); }
            else { if (stage) k_mcc<2, true><<<grid, PIC1D_NT, sm, st>>>(m); else k_mcc<2, false><<<grid, PIC1D_NT, 0, st>>>(m); }
            mark(h, "mcc", s);
        }
        if (kind == 1) {
            k_mcc_births<<<h->num_sms * 4, PIC1D_NT, 0, st>>>(m);
            mark(h, "mcc_births", s);
        }
    }
    for (int s = 0; s < c.n_species; ++s) {  // binary collisions inside the sort cells (after the MCC, like the oracle)
        if (!(c.coul_A[s] > 0.0)) continue;
        SpeciesHost& p = h->sp[s];
        CoulombArgs ca;
        ca.vx = p.buf[p.cur][1]; ca.vy = p.buf[p.cur][2]; ca.vz = p.buf[p.cur][3];
        ca.offsets = p.offsets; ca.partner = p.partner; ca.st = h->st; ca.s = s; ca.n_sc = h->n_sc;
        ca.A = (float)c.coul_A[s]; ca.k0 = (uint32_t)c.seed; ca.k1 = (uint32_t)(c.seed >> 32);
        // staging for cells of up to twice the mean count the arrays were sized for, 72 KB at most (3 blocks / SM)
        const int64_t per_cell = p.capacity / std::max(1, h->n_sc);
        ca.slots = (int)std::min<int64_t>(6144, std::max<int64_t>(1024, (2 * per_cell + 255) / 256 * 256));
        k_coulomb<<<std::min(h->n_sc, h->num_sms * 8), PIC1D_NT, (size_t)ca.slots * 12, st>>>(ca);
        mark(h, "coulomb", s);
    }
}

// the null-test bit mask of species s for the NEXT step (k_null_bits_next), once this step's scatter has used the
// current one.  Placement measured (profiles/r2_notes.md): at the end of the side stream's work, after the births.
void enqueue_null_next(pic1d* h, int s, cudaStream_t st) {
    SpeciesHost& p = h->sp[s];
    if (!p.mcck) return;
    const int n_words = p.capacity / 32;
    k_null_bits_next<<<(n_words + 255) / 256, 256, 0, st>>>(mcc_params(h, s), n_words);
    mark(h, "null_bits", s);
}

void enqueue_step(pic1d* h) {
    const pic1d_config_t& c = h->cfg;
    const bool overlap = h->side != nullptr && !h->timing && !(c.flags & PIC1D_FLAG_NO_OVERLAP);
    enqueue_begin(h, 1);
    if (c.n_species > 1) {
        enqueue_sort(h, 1, 1);
        if (h->abs_list) {
            SpeciesHost& pe = h->sp[0];
            SeeArgs sa;
            sa.st = h->st; sa.abs_list = h->abs_list; sa.abs_cap = h->abs_cap;
            sa.ex = pe.buf[pe.cur][0]; sa.evx = pe.buf[pe.cur][1]; sa.evy = pe.buf[pe.cur][2]; sa.evz = pe.buf[pe.cur][3];
            sa.cap_e = pe.capacity; sa.T = pe.T;
            sa.gamma = (float)c.see_gamma; sa.vth = (float)c.see_vth; sa.fNc = (float)c.n_cells;
            sa.k0 = (uint32_t)c.seed; sa.k1 = (uint32_t)(c.seed >> 32);
            k_see_emit<<<1, 1024, 0, h->stream>>>(sa);
            mark(h, "see_emit", 0);
        }
    }
    enqueue_sort(h, 0, 1);
    // fork: collisions + births on the side stream, deposit + field on the caller's; join at the end of the step
    if (overlap) {
        cudaEventRecord(h->ev_fork, h->stream);
        cudaStreamWaitEvent(h->side, h->ev_fork, 0);
        enqueue_mcc(h, h->side);
        for (int s = c.n_species - 1; s >= 0; --s) enqueue_null_next(h, s, h->side);
        cudaEventRecord(h->ev_join, h->side);
        enqueue_grid(h, 1);
        cudaStreamWaitEvent(h->stream, h->ev_join, 0);
    } else {
        enqueue_grid(h, 1);
        enqueue_mcc(h, h->stream);
        for (int s = c.n_species - 1; s >= 0; --s) enqueue_null_next(h, s, h->stream);
    }
    h->step += 1u;
    h->null_ready = true;
}

int sticky_code(unsigned err) {
    if (err & ERRBIT_NONFINITE) return PIC1D_ERR_NONFINITE;
    if (err & ERRBIT_CAPACITY) return PIC1D_ERR_CAPACITY;
    if (err & ERRBIT_WORKSPACE) return PIC1D_ERR_WORKSPACE;
    if (err & ERRBIT_BADLOAD) return PIC1D_ERR_ARG;
    return PIC1D_OK;
}

int fetch_state(pic1d* h, DevState* out) {
    if (!ck(h, cudaMemcpyAsync(out, h->st, sizeof(DevState), cudaMemcpyDeviceToHost, h->stream))) return PIC1D_ERR_CUDA;
    if (!ck(h, cudaStreamSynchronize(h->stream))) return PIC1D_ERR_CUDA;
    return PIC1D_OK;
}

__global__ void k_set_count(DevState* st, int s, int n) {
    DevSpecies& sp = st->sp[s];
    memset(&sp, 0, sizeof(sp));
    sp.n_live = n;
}
__global__ void k_clear_err(DevState* st) { st->err = 0; st->step = 0; st->step_next = 0; st->n_abs = 0; }

// The one exit of a handle: every CUDA object it owns (pic1d{} starts them all as null), then the handle.
void free_handle(pic1d* h) {
    for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
    for (cudaGraphExec_t g : h->graph) if (g) cudaGraphExecDestroy(g);
    if (h->side) { cudaStreamSynchronize(h->side); cudaStreamDestroy(h->side); }
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    delete h;
}

}  // namespace

// =================================== C-ABI ===========================================================
extern "C" {

int pic1d_workspace_bytes(const pic1d_config_t* cfg, size_t* bytes_out) {
    if (!bytes_out) return PIC1D_ERR_ARG;
    int rc = validate_cfg(cfg);
    if (rc) return rc;
    pic1d tmp{};
    tmp.cfg = *cfg;
    *bytes_out = layout(&tmp, nullptr);
    return PIC1D_OK;
}

int pic1d_create(const pic1d_config_t* cfg, void* workspace, size_t workspace_bytes, void* cuda_stream,
                 pic1d_t** out) {
    if (!out || !workspace) return PIC1D_ERR_ARG;
    int rc = validate_cfg(cfg);
    if (rc) return rc;
    if (reinterpret_cast<uintptr_t>(workspace) % 256 != 0) return PIC1D_ERR_ARG;
    pic1d* h = new (std::nothrow) pic1d{};
    if (!h) return PIC1D_ERR_ARG;
    h->cfg = *cfg;
    h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    const size_t need = layout(h, reinterpret_cast<char*>(workspace));
    if (need > workspace_bytes) { delete h; return PIC1D_ERR_WORKSPACE; }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        delete h;
        return PIC1D_ERR_CUDA;
    }
    h->num_sms = prop.multiProcessorCount;
    if (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        free_handle(h);
        return PIC1D_ERR_CUDA;
    }
    setup_launch(h);
    h->last_err = cudaSuccess;
    // zero the bookkeeping (state, look-back descriptors); particle arrays need no initialisation
    bool ok = ck(h, cudaMemsetAsync(h->st, 0, sizeof(DevState), h->stream));
    if (h->ion_bits) {
        ok = ok && ck(h, cudaMemsetAsync(h->ion_bits, 0, sizeof(unsigned) * h->n_ion_words, h->stream));
        ok = ok && ck(h, cudaMemsetAsync(h->ion_nb, 0, sizeof(int) * h->sp[0].n_mcc_tiles, h->stream));
    }
    ok = ok && ck(h, cudaMemsetAsync(h->E32, 0, sizeof(float) * (h->nodes + 1), h->stream));
    if (!ok || !ck(h, cudaGetLastError())) { free_handle(h); return PIC1D_ERR_CUDA; }
    *out = h;
    return PIC1D_OK;
}

int pic1d_destroy(pic1d_t* h) {
    if (!h) return PIC1D_OK;
    cudaStreamSynchronize(h->stream);
    free_handle(h);
    return PIC1D_OK;
}

int pic1d_load_particles(pic1d_t* h, int s, int64_t n, const float* x, const float* vx, const float* vy,
                         const float* vz, int on_device) {
    if (!h || s < 0 || s >= h->cfg.n_species || n < 0) return PIC1D_ERR_ARG;
    if (n > 0 && (!x || !vx || !vy || !vz)) return PIC1D_ERR_ARG;
    SpeciesHost& p = h->sp[s];
    if (n > p.capacity) return PIC1D_ERR_CAPACITY;
    if (h->loaded_mask == 0) {  // a new run starts: all species must be (re)loaded
        h->ready = false;
        h->null_ready = false;
        for (int q = 0; q < h->cfg.n_species; ++q) h->sp[q].cur = 0;
        k_clear_err<<<1, 1, 0, h->stream>>>(h->st);
        h->launches++;
    }
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    const float* src[4] = {x, vx, vy, vz};
    for (int k = 0; k < 4 && n > 0; ++k)
        if (!ck(h, cudaMemcpyAsync(p.buf[0][k], src[k], (size_t)n * sizeof(float), kind, h->stream)))
            return PIC1D_ERR_CUDA;
    k_set_count<<<1, 1, 0, h->stream>>>(h->st, s, (int)n);
    k_validate<<<(int)std::min<int64_t>(1024, n / 256 + 1), 256, 0, h->stream>>>(p.buf[0][0], (int)n, (float)h->cfg.n_cells, h->st);
    h->launches += 2;
    h->loaded_mask |= 1 << s;
    if (h->loaded_mask != (1 << h->cfg.n_species) - 1) {
        if (!ck(h, cudaGetLastError())) return PIC1D_ERR_CUDA;
        // host arrays are "copied; the caller keeps ownership": they may be reused or freed as soon as we return
        if (!on_device && !ck(h, cudaStreamSynchronize(h->stream))) return PIC1D_ERR_CUDA;
        return PIC1D_OK;
    }
    // last species in: fine-sort, deposit and solve so that rho / phi / E are valid for step 0
    h->loaded_mask = 0;
    h->step = 0;
    for (int q = 0; q < h->cfg.n_species; ++q) {
        SpeciesHost& pq = h->sp[q];
        if (pq.mask) cudaMemsetAsync(pq.mask, 0, pq.capacity, h->stream);
    }
    // An unsorted load has full-width tile windows, wider than a tile's fixed pool row.  Sort by the
    // leading bits of the sort cell first, then by more bits, ... then by the sort cell: a sequence of
    // stable passes = one stable sort, and every pass sees windows no wider than the pool row.
    int bits = 0;
    while ((1 << bits) < h->n_sc) ++bits;
    int passes[PIC1D_MAX_SPECIES], sb[PIC1D_MAX_SPECIES], rounds = 1;
    for (int q = 0; q < h->cfg.n_species; ++q) {
        sb[q] = 0;
        while ((2 << sb[q]) <= h->sp[q].pool_stride) ++sb[q];
        sb[q] = std::max(sb[q], 1);
        passes[q] = std::max(1, (bits + sb[q] - 1) / sb[q]);
        rounds = std::max(rounds, passes[q]);
    }
    for (int r = 0; r < rounds; ++r) {
        enqueue_begin(h, 0);
        for (int q = h->cfg.n_species - 1; q >= 0; --q) {
            const int pidx = r - (rounds - passes[q]);  // species with fewer passes join late
            if (pidx < 0) continue;
            enqueue_sort(h, q, 0, std::max(0, bits - (pidx + 1) * sb[q]));
        }
    }
    enqueue_grid(h, 0);
    if (!ck(h, cudaGetLastError())) return PIC1D_ERR_CUDA;
    if (!on_device && !ck(h, cudaStreamSynchronize(h->stream))) return PIC1D_ERR_CUDA;  // host buffers may go away
    h->ready = true;
    return PIC1D_OK;
}

int pic1d_step(pic1d_t* h, int n_steps) {
    if (!h || n_steps < 0 || !h->ready) return PIC1D_ERR_ARG;
    int k = 0;
    // Two consecutive steps (the sort buffers swap every step, so two steps restore the pointers) are captured
    // once per buffer parity into a CUDA graph and replayed: every per-step quantity (step index, particle
    // counts, tickets) lives in DevState on the device, no kernel argument changes from step to step.
    if (!h->null_ready && n_steps > 0) { enqueue_step(h); k = 1; }  // (a captured step counts on the masks computed ahead)
    if (!(h->cfg.flags & PIC1D_FLAG_NO_GRAPH) && !h->graph_off) {
        while (n_steps - k >= 2) {
            // the baked kernel arguments depend on which buffer of EVERY species is current
            const int par = h->sp[0].cur | (h->cfg.n_species > 1 ? h->sp[1].cur << 1 : 0);
            if (!h->graph[par]) {
                cudaGraph_t g = nullptr;
                if (cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
                    cudaGetLastError();
                    h->graph_off = true;  // e.g. the legacy default stream: do not try again every call
                    break;
                }
                const int64_t l0 = h->launches;
                const uint32_t s0 = h->step;
                enqueue_step(h);
                enqueue_step(h);
                h->launches_per_2steps = h->launches - l0;
                h->launches = l0; h->step = s0;  // captured, not run
                const cudaError_t e = cudaStreamEndCapture(h->stream, &g);
                if (e != cudaSuccess || !g || cudaGraphInstantiate(&h->graph[par], g, 0) != cudaSuccess) {
                    if (g) cudaGraphDestroy(g);
                    h->graph[par] = nullptr;
                    cudaGetLastError();
                    h->graph_off = true;
                    break;
                }
                cudaGraphDestroy(g);
            }
            if (!ck(h, cudaGraphLaunch(h->graph[par], h->stream))) return PIC1D_ERR_CUDA;
            ++h->graph_launches;
            h->launches += h->launches_per_2steps;
            h->step += 2u;
            k += 2;
        }
    }
    for (; k < n_steps; ++k) enqueue_step(h);
    return ck(h, cudaGetLastError()) ? PIC1D_OK : PIC1D_ERR_CUDA;
}

int pic1d_step_timed(pic1d_t* h, pic1d_kernel_time_t* out, int max_kernels) {
    if (!h || !out || max_kernels <= 0 || !h->ready) return PIC1D_ERR_ARG;
    h->timing = true;
    h->marks.clear();
    h->ev_used = 0;
    mark(h, "start", -1);
    h->launches--;
    enqueue_step(h);
    h->timing = false;
    if (!ck(h, cudaStreamSynchronize(h->stream))) return PIC1D_ERR_CUDA;
    int n = 0;
    for (size_t i = 1; i < h->marks.size() && n < max_kernels; ++i, ++n) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, h->marks[i - 1].ev, h->marks[i].ev);
        snprintf(out[n].name, sizeof(out[n].name), "%s", h->marks[i].name);
        out[n].ms = ms;
        out[n].species = h->marks[i].species;
    }
    return n;
}

int pic1d_get_rho_phi_E(pic1d_t* h, double* rho, double* phi, double* E, int n_nodes, int on_device) {
    if (!h || n_nodes != h->nodes || !h->ready) return PIC1D_ERR_ARG;
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    const size_t bytes = (size_t)n_nodes * sizeof(double);
    if (rho && !ck(h, cudaMemcpyAsync(rho, h->rho, bytes, kind, h->stream))) return PIC1D_ERR_CUDA;
    if (phi && !ck(h, cudaMemcpyAsync(phi, h->phi, bytes, kind, h->stream))) return PIC1D_ERR_CUDA;
    if (E && !ck(h, cudaMemcpyAsync(E, h->E, bytes, kind, h->stream))) return PIC1D_ERR_CUDA;
    if (on_device) return PIC1D_OK;
    DevState st;
    int rc = fetch_state(h, &st);
    return rc ? rc : sticky_code(st.err);
}

int pic1d_moments(pic1d_t* h, int s, pic1d_moments_t* out, double* density, int n_density, int64_t* eedf,
                  int n_bins, double E_max) {
    if (!h || !out || s < 0 || s >= h->cfg.n_species || !h->ready) return PIC1D_ERR_ARG;
    if (density && n_density != h->nodes) return PIC1D_ERR_ARG;
    if (eedf && (n_bins <= 0 || n_bins > h->eedf_cap || !(E_max > 0.0))) return PIC1D_ERR_ARG;
    SpeciesHost& p = h->sp[s];
    MomArgs m;
    m.vx = p.buf[p.cur][1]; m.vy = p.buf[p.cur][2]; m.vz = p.buf[p.cur][3];
    m.st = h->st; m.s = s; m.partial = h->mom_partial;
    m.eedf = eedf ? h->eedf_dev : nullptr; m.n_bins = n_bins; m.E_max = E_max; m.c_eV = h->cfg.sp[s].c_eV;
    if (eedf) cudaMemsetAsync(h->eedf_dev, 0, sizeof(ull) * n_bins, h->stream);
    k_moments<<<MOM_BLOCKS, 256, 0, h->stream>>>(m);
    h->launches++;
    std::vector<double> part(MOM_BLOCKS * 5);
    if (!ck(h, cudaMemcpyAsync(part.data(), h->mom_partial, sizeof(double) * MOM_BLOCKS * 5, cudaMemcpyDeviceToHost, h->stream)))
        return PIC1D_ERR_CUDA;
    if (density && !ck(h, cudaMemcpyAsync(density, p.rho_s, sizeof(double) * h->nodes, cudaMemcpyDeviceToHost, h->stream)))
        return PIC1D_ERR_CUDA;
    if (eedf && !ck(h, cudaMemcpyAsync(eedf, h->eedf_dev, sizeof(ull) * n_bins, cudaMemcpyDeviceToHost, h->stream)))
        return PIC1D_ERR_CUDA;
    DevState st;
    int rc = fetch_state(h, &st);
    if (rc) return rc;
    double acc[5] = {0, 0, 0, 0, 0};
    for (int b = 0; b < MOM_BLOCKS; ++b)
        for (int k = 0; k < 5; ++k) acc[k] += part[b * 5 + k];
    const DevSpecies& d = st.sp[s];
    memset(out, 0, sizeof(*out));
    out->count = d.n_live; out->n_sorted = d.n_sorted;
    out->sum_vx = acc[0]; out->sum_vy = acc[1]; out->sum_vz = acc[2]; out->sum_v2 = acc[3]; out->sum_v4 = acc[4];
    out->absorbed_left = (int64_t)d.absorbed_left; out->absorbed_right = (int64_t)d.absorbed_right;
    out->injected = (int64_t)d.injected; out->n_candidates = (int64_t)d.n_candidates;
    for (int k = 0; k < 4; ++k) out->n_events[k] = (int64_t)d.n_events[k];
    out->births = (int64_t)d.births; out->dropped = (int64_t)d.dropped; out->over_cap = (int64_t)d.over_cap;
    out->reflected = (int64_t)d.reflected; out->n_pairs = (int64_t)d.n_pairs;
    return sticky_code(st.err);
}

int pic1d_n_nodes(const pic1d_t* h) { return h ? h->nodes : PIC1D_ERR_ARG; }
int pic1d_n_sort_cells(const pic1d_t* h) { return h ? h->n_sc : PIC1D_ERR_ARG; }
uint32_t pic1d_step_index(const pic1d_t* h) { return h ? h->step : 0u; }
const char* pic1d_last_cuda_error(const pic1d_t* h) { return h ? cudaGetErrorString(h->last_err) : "null handle"; }
int pic1d_abi_version(void) { return PIC1D_ABI_VERSION; }
int64_t pic1d_launch_count(const pic1d_t* h) { return h ? h->launches : 0; }
int64_t pic1d_graph_launch_count(const pic1d_t* h) { return !h ? 0 : h->graph_off ? -1 : h->graph_launches; }

int pic1d_debug_count(pic1d_t* h, int what, int s, int64_t* count_out) {
    if (!h || !count_out || s < 0 || s >= h->cfg.n_species || !h->ready) return PIC1D_ERR_ARG;
    DevState st;
    int rc = fetch_state(h, &st);
    if (rc) return rc;
    switch (what) {
        case PIC1D_DBG_X: case PIC1D_DBG_VX: case PIC1D_DBG_VY: case PIC1D_DBG_VZ: *count_out = st.sp[s].n_live; break;
        case PIC1D_DBG_KEYS: *count_out = st.sp[s].n_src; break;
        case PIC1D_DBG_OFFSETS: *count_out = h->n_sc + 1; break;
        case PIC1D_DBG_MASK: case PIC1D_DBG_PARTNER: *count_out = st.sp[s].n_sorted; break;
        case PIC1D_DBG_E32: case PIC1D_DBG_RHO_S: *count_out = h->nodes; break;
        case PIC1D_DBG_TILE_W: *count_out = st.sp[s].n_tiles; break;
        default: return PIC1D_ERR_ARG;
    }
    return PIC1D_OK;
}

int pic1d_debug_get(pic1d_t* h, int what, int s, void* dst, size_t bytes) {
    int64_t n = 0;
    int rc = pic1d_debug_count(h, what, s, &n);
    if (rc) return rc;
    if (!dst) return PIC1D_ERR_ARG;
    SpeciesHost& p = h->sp[s];
    const void* src = nullptr;
    size_t el = 4;
    switch (what) {
        case PIC1D_DBG_X: case PIC1D_DBG_VX: case PIC1D_DBG_VY: case PIC1D_DBG_VZ: src = p.buf[p.cur][what]; break;
        case PIC1D_DBG_KEYS: src = p.keys_dbg; break;
        case PIC1D_DBG_OFFSETS: src = p.offsets; break;
        case PIC1D_DBG_MASK: src = p.mask; el = 1; break;
        case PIC1D_DBG_E32: src = h->E32; break;
        case PIC1D_DBG_RHO_S: src = p.rho_s; el = 8; break;
        case PIC1D_DBG_TILE_W: src = p.tile_w; break;
        case PIC1D_DBG_PARTNER: src = p.partner; break;
    }
    if (!src || bytes < (size_t)n * el) return PIC1D_ERR_ARG;
    if (n > 0 && !ck(h, cudaMemcpyAsync(dst, src, (size_t)n * el, cudaMemcpyDeviceToHost, h->stream))) return PIC1D_ERR_CUDA;
    return ck(h, cudaStreamSynchronize(h->stream)) ? PIC1D_OK : PIC1D_ERR_CUDA;
}

__global__ void k_debug_set_counts(DevState* st, int s, int n_live, int n_sorted, int set_step, unsigned step) {
    st->sp[s].n_live = n_live;
    st->sp[s].n_sorted = n_sorted;
    if (set_step) st->step_next = step;
}

int pic1d_debug_set_state(pic1d_t* h, int s, int64_t n, int64_t n_sorted, const float* x, const float* vx,
                          const float* vy, const float* vz, int64_t step) {
    if (!h || s < 0 || s >= h->cfg.n_species || !h->ready || n < 0 || n_sorted < 0 || n_sorted > n) return PIC1D_ERR_ARG;
    SpeciesHost& p = h->sp[s];
    if (n > p.capacity) return PIC1D_ERR_CAPACITY;
    const float* src[4] = {x, vx, vy, vz};
    for (int k = 0; k < 4 && n > 0; ++k)
        if (!src[k] || !ck(h, cudaMemcpyAsync(p.buf[p.cur][k], src[k], (size_t)n * sizeof(float), cudaMemcpyHostToDevice, h->stream)))
            return PIC1D_ERR_CUDA;
    k_debug_set_counts<<<1, 1, 0, h->stream>>>(h->st, s, (int)n, (int)n_sorted, step >= 0 ? 1 : 0, (unsigned)(step >= 0 ? step : 0));
    if (step >= 0) h->step = (uint32_t)step;
    h->null_ready = false;  // the masks enqueued ahead belong to another step index / another particle count
    return ck(h, cudaStreamSynchronize(h->stream)) ? PIC1D_OK : PIC1D_ERR_CUDA;
}

int pic1d_debug_set_E32(pic1d_t* h, const float* E32, int n_nodes) {
    if (!h || !E32 || n_nodes != h->nodes) return PIC1D_ERR_ARG;
    if (!ck(h, cudaMemcpyAsync(h->E32, E32, sizeof(float) * n_nodes, cudaMemcpyHostToDevice, h->stream))) return PIC1D_ERR_CUDA;
    return ck(h, cudaStreamSynchronize(h->stream)) ? PIC1D_OK : PIC1D_ERR_CUDA;
}

}  // extern "C"
