// pic1d_grid.cuh -- charge deposition over the sorted per-cell ranges (Fig. 4-5),
// the edge-node follow-up kernel (L138) and the single-block Poisson + E solve (Eq. 1-2,
// L142-146).  fp64 throughout; no global floating-point atomics anywhere.
#pragma once
#include "pic1d_device.cuh"

struct DepositSpecies {
    const float* x;      // sorted positions of the species
    const int* offsets;  // [n_sc + 1]
    double* part;        // [n_blocks * G]   nodes c0 .. c1-1 of each block (left-closed)
    double* side;        // [n_blocks]       right edge node c1 of each block (paper's side array, L138)
};
struct DepositArgs {
    DepositSpecies sp[2];  // blockIdx.y = species: one launch deposits every species
    int Nc, n_sc, G;       // G grid cells per block (a multiple of the sort-cell size when r > 1)
    float inv_r;
};

__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Block b owns grid cells [b G, (b+1) G) and therefore the contiguous slot range
// offsets[key(b G)] .. offsets[key((b+1) G)] of the sorted array; every warp takes a contiguous part
// of it.  The node weights are accumulated as 64-bit FIXED-POINT integers in units of 2^-40: f = x - j
// is a multiple of 2^-23 for x >= 1, so the integer sums are exact and equal, after conversion, to the
// oracle's fp64 sums in any order (sums stay below 2^53 for up to 8192 particles per node; only
// particles with x < 2^-17 lose bits, below the rounding of the fp64 sum itself).  While a warp's rows
// stay in one cell the per-lane sums live in registers (the paper's register partial sums, L130) and
// are reduced with shuffles when the cell changes; rows that straddle cells are split by cell value, one
// warp reduction per distinct cell.
#define DEP_ONE (1ll << 40)
#define DEP_U 4  // rows in flight per warp

__device__ __forceinline__ long long warp_sum_ll(long long v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

struct DepAcc {  // a warp's register partial sums for its current cell
    int jc, accn;
    long long accF;
};

__device__ __forceinline__ void dep_flush(DepAcc& A, ull* s_acc, int c0, int lane) {
    if (A.jc >= 0) {
        const long long Fs = warp_sum_ll(A.accF);
        const int n = __reduce_add_sync(0xffffffffu, A.accn);
        if (lane == 0) {
            atomicAdd(&s_acc[A.jc - c0], (ull)((long long)n * DEP_ONE - Fs));
            atomicAdd(&s_acc[A.jc + 1 - c0], (ull)Fs);
        }
    }
    A.accF = 0; A.accn = 0;
}

// one row of 32 slots (one particle per lane).  A row that straddles cells (every row when a sort cell
// holds several grid cells, r > 1) adds its two weights per lane as three 14-bit limbs with native 32-bit
// shared reductions (conflicting red.shared is not serialised on sm_100a); `limbs` is off when the block
// holds so many particles that a limb counter could overflow (2^18 additions), then the row is split by
// cell value with one warp reduction per distinct cell.
#define DEP_LIMB_MAX 200000
__device__ __forceinline__ void dep_limbs(unsigned* s_l, int node, int np1, long long v) {
    atomicAdd(&s_l[node], (unsigned)(v & 0x3fff));
    atomicAdd(&s_l[np1 + node], (unsigned)((v >> 14) & 0x3fff));
    atomicAdd(&s_l[2 * np1 + node], (unsigned)(v >> 28));
}

__device__ __forceinline__ void dep_row(bool valid, float xv, DepAcc& A, ull* s_acc, unsigned* s_l, int np1,
                                        bool limbs, int c0, int lane) {
    const int j = (int)xv;
    const long long F = __float2ll_rz(__fmul_rn(__fsub_rn(xv, (float)j), 0x1p40f));
    const int j0 = __shfl_sync(0xffffffffu, j, 0);
    if (__all_sync(0xffffffffu, valid && j == j0)) {
        if (j0 != A.jc) { dep_flush(A, s_acc, c0, lane); A.jc = j0; }
        A.accF += F; ++A.accn;
    } else if (limbs) {
        if (valid) {
            dep_limbs(s_l, j - c0, np1, DEP_ONE - F);
            dep_limbs(s_l, j + 1 - c0, np1, F);
        }
    } else {  // one warp reduction per distinct cell
        unsigned rem = __ballot_sync(0xffffffffu, valid);
        while (rem) {
            const int jj = __shfl_sync(0xffffffffu, j, __ffs(rem) - 1);
            const bool in = valid && j == jj;
            const unsigned grp = __ballot_sync(0xffffffffu, in);
            const long long Fs = warp_sum_ll(in ? F : 0ll);
            if (lane == 0) {
                atomicAdd(&s_acc[jj - c0], (ull)((long long)__popc(grp) * DEP_ONE - Fs));
                atomicAdd(&s_acc[jj + 1 - c0], (ull)Fs);
            }
            rem &= ~grp;
        }
    }
}

__global__ void __launch_bounds__(PIC1D_NT) k_deposit(DepositArgs args) {
    extern __shared__ ull s_acc[];  // G + 1 nodes, then 3 x (G + 1) 32-bit limb counters
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    struct { const float* x; const int* offsets; double* part; double* side; int Nc, n_sc, G; float inv_r; } a;
    a.x = args.sp[blockIdx.y].x; a.offsets = args.sp[blockIdx.y].offsets; a.part = args.sp[blockIdx.y].part;
    a.side = args.sp[blockIdx.y].side; a.Nc = args.Nc; a.n_sc = args.n_sc; a.G = args.G; a.inv_r = args.inv_r;
    const int c0 = blockIdx.x * a.G, c1 = min(c0 + a.G, a.Nc);
    const int k0 = (int)__fmul_rn((float)c0, a.inv_r);
    const int k1 = c1 >= a.Nc ? a.n_sc : (int)__fmul_rn((float)c1, a.inv_r);
    const int p0 = a.offsets[k0], p1 = a.offsets[k1];
    const int np1 = a.G + 1;
    unsigned* s_l = reinterpret_cast<unsigned*>(s_acc + np1);
    const bool limbs = p1 - p0 <= DEP_LIMB_MAX;  // block-uniform
    for (int i = tid; i <= a.G; i += PIC1D_NT) { s_acc[i] = 0ull; s_l[i] = 0u; s_l[np1 + i] = 0u; s_l[2 * np1 + i] = 0u; }
    __syncthreads();
    // [p0, p1) = head [p0, a0) + 128-slot chunks [a0, a1) + tail [a1, p1); chunks are read as float4
    const int a0 = min(p1, (p0 + 127) & ~127), a1 = max(a0, p1 & ~127);
    DepAcc A;
    A.jc = -1; A.accn = 0; A.accF = 0;
    if (wp == 0) {  // head and tail, row by row
        for (int i0 = p0; i0 < a0; i0 += 32) {
            const int i = i0 + lane;
            dep_row(i < a0, i < a0 ? __ldcs(a.x + i) : 0.0f, A, s_acc, s_l, np1, limbs, c0, lane);
        }
        for (int i0 = a1; i0 < p1; i0 += 32) {
            const int i = i0 + lane;
            dep_row(i < p1, i < p1 ? __ldcs(a.x + i) : 0.0f, A, s_acc, s_l, np1, limbs, c0, lane);
        }
    }
    const int ch_w = ((a1 - a0) / 128 + PIC1D_NWARP - 1) / PIC1D_NWARP;  // chunks per warp
    const int cb = min(a0 + wp * ch_w * 128, a1), ce = min(cb + ch_w * 128, a1);
    for (int i0 = cb; i0 < ce; i0 += 128 * DEP_U) {
        float4 q[DEP_U];
#pragma unroll
        for (int u = 0; u < DEP_U; ++u)
            if (i0 + u * 128 < ce) q[u] = __ldcs(reinterpret_cast<const float4*>(a.x + i0 + u * 128) + lane);
#pragma unroll
        for (int u = 0; u < DEP_U; ++u) {
            if (i0 + u * 128 >= ce) break;  // warp-uniform
            const int jx = (int)q[u].x, jy = (int)q[u].y, jz = (int)q[u].z, jw = (int)q[u].w;
            const int j0 = __shfl_sync(0xffffffffu, jx, 0);
            if (__all_sync(0xffffffffu, (jx == j0) & (jy == j0) & (jz == j0) & (jw == j0))) {
                if (j0 != A.jc) { dep_flush(A, s_acc, c0, lane); A.jc = j0; }
                const float fj = (float)j0;
                A.accF += __float2ll_rz(__fmul_rn(__fsub_rn(q[u].x, fj), 0x1p40f)) +
                          __float2ll_rz(__fmul_rn(__fsub_rn(q[u].y, fj), 0x1p40f)) +
                          __float2ll_rz(__fmul_rn(__fsub_rn(q[u].z, fj), 0x1p40f)) +
                          __float2ll_rz(__fmul_rn(__fsub_rn(q[u].w, fj), 0x1p40f));
                A.accn += 4;
            } else {  // the chunk straddles cells
                dep_row(true, q[u].x, A, s_acc, s_l, np1, limbs, c0, lane); dep_row(true, q[u].y, A, s_acc, s_l, np1, limbs, c0, lane);
                dep_row(true, q[u].z, A, s_acc, s_l, np1, limbs, c0, lane); dep_row(true, q[u].w, A, s_acc, s_l, np1, limbs, c0, lane);
            }
        }
    }
    dep_flush(A, s_acc, c0, lane);
    __syncthreads();
    auto node = [&](int i) {
        return (double)(s_acc[i] + (ull)s_l[i] + ((ull)s_l[np1 + i] << 14) + ((ull)s_l[2 * np1 + i] << 28)) * 0x1p-40;
    };
    for (int i = tid; i < a.G; i += PIC1D_NT) a.part[(size_t)blockIdx.x * a.G + i] = node(i);
    if (tid == 0) a.side[blockIdx.x] = node(c1 - c0);
}

// Follow-up step (L138; here the prologue of the field kernel, not a launch of its own): node j of species s =
// block part + the left neighbour's right-edge node; net rho = background + sum_s sign_s rho_s.
struct CombineArgs {
    const double* part[2];
    const double* side[2];
    double* rho_s[2];
    double* rho;
    int sign[2];
    int n_species, Nc, nodes, G, bc;
    double background;
};

__device__ __forceinline__ void rho_combine_node(const CombineArgs& a, int j) {
    const int nb = (a.Nc + a.G - 1) / a.G;
    double r = a.background;
    for (int s = 0; s < a.n_species; ++s) {
        double v = j < a.Nc ? a.part[s][j] : 0.0;  // part is indexed by node because blocks are G-aligned
        if (j == a.Nc) v += a.side[s][nb - 1];               // bounded: right wall node
        else if (j > 0 && j % a.G == 0) v += a.side[s][j / a.G - 1];
        if (a.bc == 1 && j == 0) v += a.side[s][nb - 1];     // periodic: node N_c == node 0
        a.rho_s[s][j] = v;
        r += (double)a.sign[s] * v;
    }
    a.rho[j] = r;
}

// ---- Poisson + E, one block --------------------------------------------------------------------
// The tridiagonal system  phi[j-1] - 2 phi[j] + phi[j+1] = -rho[j]  (Eq. 1 discretised, L142) with
// Dirichlet ends has the closed solution
//     d_j = phi_j - phi_{j-1} = d_1 - S_{j-1},   S_m = sum_{i=1..m} rho_i,
//     phi_j = phi_0 + j d_1 - T_{j-1},           T_m = sum_{i=1..m} S_i,
//     d_1 = (phi_N - phi_0 + T_{N-1}) / N,
// i.e. the Thomas recurrences (L142) summed in closed form, which turns the serial elimination into
// two block-wide fp64 prefix sums.  E_j = (phi_{j-1} - phi_{j+1}) / 2 = -d_1 + (S_{j-1} + S_j) / 2.
struct FieldArgs {
    CombineArgs cb;  // the deposit's partial sums -> rho_s, rho (prologue)
    const double* rho;
    double *phi, *E, *S, *Tt;
    float* E32;
    int Nc, nodes, bc;
    double V0, omega_dt;
    const DevState* st;  // in_step: the wall potential is taken at t_{n+1}, n = st->step (device-resident)
    int in_step;         // 0: t = 0 (right after a load)
};

__device__ double block_sum_d(double v) {
    __shared__ double s_r[32];
    __shared__ double s_out;
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    v = warp_sum_d(v);
    if (lane == 0) s_r[wp] = v;
    __syncthreads();
    if (wp == 0) {
        double t = lane < (blockDim.x >> 5) ? s_r[lane] : 0.0;
        t = warp_sum_d(t);
        if (lane == 0) s_out = t;
    }
    __syncthreads();
    const double r = s_out;
    __syncthreads();
    return r;
}

// inclusive scan of n doubles, dst[i] = sum_{m<=i} src(m); thread-contiguous chunks.
template <class F>
__device__ void block_inclusive_scan_d(F src, double* dst, int n) {
    __shared__ double s_w[32];
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5, nw = blockDim.x >> 5;
    const int ch = (n + blockDim.x - 1) / blockDim.x;
    const int b = tid * ch, e = min(b + ch, n);
    double tot = 0.0;
    for (int i = b; i < e; ++i) tot += src(i);
    double inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        double t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[wp] = inc;
    __syncthreads();
    if (wp == 0) {
        double t = lane < nw ? s_w[lane] : 0.0, ti = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            double u = __shfl_up_sync(0xffffffffu, ti, o);
            if (lane >= o) ti += u;
        }
        s_w[lane] = ti - t;
    }
    __syncthreads();
    double run = s_w[wp] + inc - tot;
    for (int i = b; i < e; ++i) { run += src(i); dst[i] = run; }
    __syncthreads();
}

__global__ void __launch_bounds__(1024) k_field(FieldArgs a) {
    const int N = a.Nc, tid = threadIdx.x;
    for (int j = tid; j < a.nodes; j += blockDim.x) rho_combine_node(a.cb, j);
    __syncthreads();
    double mean = 0.0;
    if (a.bc == 1) {
        double p = 0.0;
        for (int i = tid; i < N; i += blockDim.x) p += a.rho[i];
        mean = block_sum_d(p) / (double)N;
    }
    const double* rho = a.rho;
    // S_j, j = 0..N-1 (S_0 = 0); T_j likewise
    block_inclusive_scan_d([=](int i) { return i == 0 ? 0.0 : rho[i] - mean; }, a.S, N);
    const double* S = a.S;
    block_inclusive_scan_d([=](int i) { return S[i]; }, a.Tt, N);
    const double phi0 = a.bc == 0 ? a.V0 * sin(a.omega_dt * (double)(a.in_step ? a.st->step + 1u : 0u)) : 0.0;
    const double phiN = 0.0;
    const double d1 = (phiN - phi0 + a.Tt[N - 1]) / (double)N;
    double psum = 0.0;
    for (int j = tid; j < a.nodes; j += blockDim.x) {
        double phi, E;
        if (j == 0) {
            phi = phi0;
            E = a.bc == 0 ? -d1 - rho[0] : -d1 + 0.5 * S[N - 1];
        } else if (j == N) {  // bounded only
            phi = phiN;
            E = -d1 + S[N - 1] + rho[N];
        } else {
            phi = phi0 + (double)j * d1 - a.Tt[j - 1];
            E = -d1 + 0.5 * (S[j - 1] + S[j]);
        }
        a.phi[j] = phi;
        a.E[j] = E;
        a.E32[j] = (float)E;
        psum += phi;
    }
    if (a.bc == 1) {  // report phi with its mean removed
        const double pm = block_sum_d(psum) / (double)N;
        for (int j = tid; j < N; j += blockDim.x) a.phi[j] -= pm;
    }
}

// Shared-memory variant for N_c <= FIELD_SMEM_MAX cells (all BASELINE configs): rho is read once,
// coalesced, into shared memory; each warp scans a contiguous segment row by row with shuffles (no bank
// conflicts, no dependent global loads); T is never stored -- phi and E are emitted while the second scan
// runs.  One launch, ~10 us at 16384 cells.
#define FIELD_SMEM_MAX 24576

__device__ __forceinline__ double warp_incl_scan_d(double v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

__global__ void __launch_bounds__(1024) k_field_smem(FieldArgs a) {
    extern __shared__ double s_S[];  // [32 * seg]
    __shared__ double s_w[32];
    const int N = a.Nc, tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    const int seg = ((N + 1023) / 1024) * 32;  // elements per warp, a multiple of 32
    const double* rho = a.rho;
    for (int j = tid; j < a.nodes; j += 1024) rho_combine_node(a.cb, j);
    __syncthreads();
    double mean = 0.0;
    if (a.bc == 1) {
        double p = 0.0;
        for (int i = tid; i < N; i += 1024) p += rho[i];
        mean = block_sum_d(p) / (double)N;
    }
    for (int i = tid; i < 32 * seg; i += 1024) s_S[i] = (i == 0 || i >= N) ? 0.0 : rho[i] - mean;
    __syncthreads();
    // scan 1: S_j = sum_{i<=j} (rho_i - mean), S_0 = 0
    const int b = wp * seg;
    {
        double carry = 0.0;
        for (int r = 0; r < seg; r += 32) {
            const double v = warp_incl_scan_d(s_S[b + r + lane], lane) + carry;
            s_S[b + r + lane] = v;
            carry = __shfl_sync(0xffffffffu, v, 31);
        }
        if (lane == 0) s_w[wp] = carry;
    }
    __syncthreads();
    {
        double off = 0.0;
        for (int q = 0; q < wp; ++q) off += s_w[q];
        __syncthreads();
        double tot = 0.0;
        for (int r = 0; r < seg; r += 32) {
            const double v = s_S[b + r + lane] + off;
            s_S[b + r + lane] = v;
            tot += (b + r + lane < N) ? v : 0.0;
        }
        tot = warp_sum_d(tot);  // sum of S over the warp's segment (elements < N)
        if (lane == 0) s_w[wp] = tot;
    }
    __syncthreads();
    // scan 2 (T_j = sum_{i<=j} S_i) fused with the outputs
    double toff = 0.0, T_all = 0.0;
    for (int q = 0; q < 32; ++q) { const double v = s_w[q]; if (q < wp) toff += v; T_all += v; }
    const double phi0 = a.bc == 0 ? a.V0 * sin(a.omega_dt * (double)(a.in_step ? a.st->step + 1u : 0u)) : 0.0;
    const double phiN = 0.0;
    const double d1 = (phiN - phi0 + T_all) / (double)N;  // T_all = T_{N-1}
    double psum = 0.0, carry = toff;
    for (int r = 0; r < seg; r += 32) {
        const int i = b + r + lane;  // element i gives node j = i + 1
        const double Si = s_S[i];
        const double Ti = warp_incl_scan_d(i < N ? Si : 0.0, lane) + carry;
        carry = __shfl_sync(0xffffffffu, Ti, 31);
        const int j = i + 1;
        if (j < N) {
            const double phi = phi0 + (double)j * d1 - Ti;
            const double E = -d1 + 0.5 * (Si + s_S[j]);
            a.phi[j] = phi; a.E[j] = E; a.E32[j] = (float)E;
            psum += phi;
        }
    }
    if (tid == 0) {
        const double SN1 = s_S[N - 1];
        const double E0 = a.bc == 0 ? -d1 - rho[0] : -d1 + 0.5 * SN1;
        a.phi[0] = phi0; a.E[0] = E0; a.E32[0] = (float)E0;
        psum += phi0;
        if (a.bc == 0) {
            const double EN = -d1 + SN1 + rho[N];
            a.phi[N] = phiN; a.E[N] = EN; a.E32[N] = (float)EN;
        }
    }
    if (a.bc == 1) {  // report phi with its mean removed
        const double pm = block_sum_d(psum) / (double)N;
        for (int j = tid; j < N; j += 1024) a.phi[j] -= pm;
    }
}

// ---- moments (diagnostic, not on the step path) ------------------------------------------------------
struct MomArgs {
    const float *vx, *vy, *vz;
    const DevState* st;
    int s;
    double* partial;  // [gridDim.x * 5]
    ull* eedf;
    int n_bins;
    double E_max, c_eV;
};

__global__ void __launch_bounds__(256) k_moments(MomArgs a) {
    const int n = a.st->sp[a.s].n_live;
    double sx = 0, sy = 0, sz = 0, s2 = 0, s4 = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const double vx = a.vx[i], vy = a.vy[i], vz = a.vz[i];
        const double g2 = (vx * vx + vy * vy) + vz * vz;
        sx += vx; sy += vy; sz += vz; s2 += g2; s4 += g2 * g2;
        if (a.eedf) {
            const double En = a.c_eV * g2;
            if (En < a.E_max) {
                const int b = (int)(En / a.E_max * (double)a.n_bins);
                if (b >= 0 && b < a.n_bins) atomicAdd(&a.eedf[b], 1ull);
            }
        }
    }
    sx = block_sum_d(sx); sy = block_sum_d(sy); sz = block_sum_d(sz);
    s2 = block_sum_d(s2); s4 = block_sum_d(s4);
    if (threadIdx.x == 0) {
        double* p = a.partial + blockIdx.x * 5;
        p[0] = sx; p[1] = sy; p[2] = sz; p[3] = s2; p[4] = s4;
    }
}

// device-side validation of freshly loaded positions: x in [0, N_c)
__global__ void k_validate(const float* x, int n, float fNc, DevState* st) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float v = x[i];
        if (!(v >= 0.0f && v < fNc)) atomicOr(&st->err, ERRBIT_BADLOAD);
    }
}
