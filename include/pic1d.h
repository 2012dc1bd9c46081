/*
 * pic1d.h -- C-ABI of the B200-native 1D3V electrostatic PIC/MCC hot path with per-cell fine
 * sorting (Mertmann et al., arXiv:1104.3998; citations are PAPER.md lines).
 *
 * One handle = one simulation on one GPU.  All device memory is a single caller-owned workspace
 * (e.g. a torch.empty(uint8) tensor); the library never allocates device memory.  All kernels are
 * enqueued on the caller's stream.  A handle is used by one host thread at a time.  Every function
 * returns 0 on success or a negative PIC1D_ERR_* code; no C++ types or exceptions cross the boundary.
 *
 * Units are the paper's normalised units (section 3.3): x in grid cells, t in steps,
 * v in cells/step, rho in super-particle charges per cell, phi in Q dx/(eps0 A_e), E in Q/(eps0 A_e).
 *
 * One call of pic1d_step(h, 1) is one pass of the cycle of Fig. 1 (L35-41), entered at the pusher:
 *   gather + leapfrog push (L35, L150-156, Eq. 3-4)  ->  wall absorption / secondary emission /
 *   compaction (L41)  ->  fine sort by sort cell (L63-67, L160-192)  ->  charge deposition over the
 *   sorted ranges (L128-138)  ->  Poisson + E (Eq. 1-2)  ->  null-collision MCC (L196-209).
 */
#ifndef PIC1D_H_
#define PIC1D_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIC1D_MAX_SPECIES 2

/* Version of this boundary: bumped whenever a struct layout, a flag, an error code or an entry point changes.
 * 3 = round 3 (pic1d_graph_launch_count, pic1d_abi_version, validation of e_reflect / coul_A; the names
 * PIC1D_FLAG_VERIFY_ORDER and PIC1D_ERR_ORDER below are retired -- kept so that callers written against
 * version 2 still compile; the library ignores the flag and never returns the code).  pic1d_abi_version()
 * returns the value the loaded library was built with: compare it with this macro after dlopen. */
#define PIC1D_ABI_VERSION 3

#define PIC1D_OK 0
#define PIC1D_ERR_ARG (-1)       /* bad argument / bad struct_size / call order */
#define PIC1D_ERR_CAPACITY (-2)  /* sticky: a load, a birth or an injection exceeded a capacity;   \
                                    the extra particles were dropped and counted */
#define PIC1D_ERR_CUDA (-3)      /* a CUDA call failed; see pic1d_last_cuda_error */
#define PIC1D_ERR_NONFINITE (-4) /* sticky: a NaN position was seen (treated as absorbed) */
#define PIC1D_ERR_WORKSPACE (-5) /* workspace too small / sort bookkeeping pool exhausted (sticky) */
#define PIC1D_ERR_ORDER (-6)     /* retired (never returned): the scatter ranks by construction now */

/* flags */
#define PIC1D_FLAG_CAPTURE 1u /* keep per-slot pre-sort keys and MCC event masks for pic1d_debug_get */
#define PIC1D_FLAG_VERIFY_ORDER 2u /* retired, ignored: every in-tile rank of the scatter now comes from match.any
                                      groups in slot order, so there is no hardware ordering left to verify */
#define PIC1D_FLAG_EQ5_ELECTRONS 4u /* hint: the electrons obey Eq. 5 (L162: they move less than about one sort
                                       cell per step), so they take the barrier-free warp-tile sort like the
                                       ions.  A performance hint within the displacement limits below. */
/*
 * Displacement limits of the fine sort.  The sort keeps, per tile of consecutive source slots, one counter per
 * sort cell of the tile's key WINDOW (lowest to highest key after the push).  Each tile owns a fixed row of
 * counters -- 32 sort cells for the warp-tile family (256 slots per tile: ions, electrons with the Eq. 5 hint),
 * min(N_sc, 4096) for the block-tile family (2048 or 1024 slots per tile: electrons) -- and wider windows draw
 * from an overflow region of max(4 Mi, capacity) counters per species.  Both families are exact for ANY
 * displacement as long as that region lasts: the windows beyond the fixed rows may sum to `capacity` sort cells,
 * i.e. on average 256 + 32 sort cells per warp tile (thermal displacement up to about 48 sort cells per step) and
 * 2048 + 4096 per block tile.  If it runs out, the tiles that got no counters are LOST: their particles are
 * counted in pic1d_moments_t.dropped and the sticky error PIC1D_ERR_WORKSPACE is raised -- the run is invalid
 * from that step on (clear the Eq. 5 hint, or raise the species' capacity).  An unsorted load never needs the
 * overflow region (it is sorted by leading key bits first).
 */
/* Where the Monte-Carlo collisions of a species run (same results either way).  Default: folded into the
 * scatter of its fine sort when its null-collision probability P0 <= 0.25 (sparse candidates), as a pass of
 * its own after the field solve (k_mcc) otherwise. */
#define PIC1D_FLAG_NO_FOLD 8u   /* never fold: every species gets the pass of its own */
#define PIC1D_FLAG_FOLD_ALL 16u /* always fold */
#define PIC1D_FLAG_MCC_GATHER 32u /* k_mcc fetches candidates' velocities with gathered loads even when most particles
                                     are candidates (default then: bulk async copies of the tile into shared memory) */

#define PIC1D_FLAG_NO_OVERLAP 64u /* run the collisions after the field solve on the caller's stream instead of beside
                                    the deposit and the field solve on an internal side stream */
#define PIC1D_FLAG_NO_GRAPH 128u  /* pic1d_step launches every kernel itself instead of replaying a captured CUDA graph
                                     of two steps (a graph needs a capturable stream: not the legacy default stream) */

typedef struct pic1d pic1d_t; /* opaque */

typedef struct pic1d_species_config {
    double kappa;       /* signed push constant kappa_s = sign(q) Q^2 dt^2/(eps0 dx M A_e), Eq. 3 (L119) */
    double c_eV;        /* eV per (cell/step)^2: E = c_eV |v|^2 */
    double P0;          /* null-collision probability P0 = 1 - exp(-dt nu_0), Eq. 6 (L200) */
    double inv_g_cap;   /* 1/g_cap [steps/cell]; g_cap = speed at which nu(g) reaches nu_0 */
    int64_t capacity;   /* slots per particle array; state + sort buffer are sized from it */
    int32_t charge_sign; /* +1 / -1 */
    int32_t mcc_kind;   /* 0 none, 1 electron set (elastic, excitation, ionisation), 2 ion charge exchange */
} pic1d_species_config_t;

typedef struct pic1d_config {
    uint32_t struct_size; /* = sizeof(pic1d_config_t) */
    int32_t n_cells;      /* N_c grid cells; bounded: N_c + 1 nodes, periodic: N_c nodes */
    int32_t bc;           /* 0 bounded with absorbing walls, 1 periodic */
    int32_t n_species;    /* 1 or 2; species 0 = electrons, species 1 = ions */
    pic1d_species_config_t sp[PIC1D_MAX_SPECIES];
    double background_rho; /* fixed neutralising background added to rho (periodic runs) */
    double sort_inv_ratio; /* 1/r, r = sort-cell size / grid-cell size, a power of two (L65, L215) */
    double V0_norm;        /* wall potential phi_0(t) = V0_norm sin(omega_dt * n); phi_{N_c} = 0 */
    double omega_dt;
    double see_gamma;      /* secondary-electron yield per absorbed ion (L41) */
    double see_vth;        /* thermal speed of emitted electrons [cells/step] */
    double r_el, r_exc, r_ion; /* sigma_el, sigma_exc0, sigma_ion0 over sigma_cap */
    double E_exc, E_ion;   /* thresholds [eV] */
    double gas_vth_ion;    /* thermal speed of the background gas for ion products [cells/step] */
    double mass_ratio;     /* m_e / M */
    uint64_t seed;         /* Philox key */
    uint32_t flags;        /* PIC1D_FLAG_* */
    uint32_t pad_;
    double e_reflect;      /* probability that an electron reaching a wall is reflected instead of absorbed: mirror
                              position, vx reversed, place in the order kept (L41: "If ... electron reflection are
                              featured, electrons are inserted at the boundaries"); 0 = off */
    double coul_A[PIC1D_MAX_SPECIES]; /* binary Coulomb collisions between the like particles of a sort cell (L69, L75,
                              L221, L259; Takizuka-Abe): <tan^2(theta/2)> = coul_A n_cell / u^3 with u in cells/step,
                              coul_A = q^4 w lnLambda dt / (8 pi eps0^2 m_r^2 A_e r dx) (dt/dx)^3, m_r = m/2; 0 = off.
                              Pairing: a keyed pseudo-random permutation of the cell's sorted slots, new every step,
                              consecutive images are partners; in a cell with an odd count one particle sits the step
                              out (Takizuka-Abe instead collide the first three among themselves) */
} pic1d_config_t;

typedef struct pic1d_moments {
    int64_t count;    /* live particles N_s (sorted part + this step's birth tail) */
    int64_t n_sorted; /* sorted part */
    double sum_vx, sum_vy, sum_vz, sum_v2, sum_v4; /* fp64 sums over all live particles */
    int64_t absorbed_left, absorbed_right;        /* cumulative since load */
    int64_t injected;     /* cumulative secondary electrons injected into this species */
    int64_t n_candidates; /* cumulative particles that passed the null test (Eq. 6) */
    int64_t n_events[4];  /* cumulative [0] null, [1] elastic or CX, [2] excitation, [3] ionisation */
    int64_t births;       /* cumulative ionisation births appended to this species */
    int64_t dropped;      /* cumulative births / injections dropped for lack of capacity */
    int64_t over_cap;     /* cumulative candidates with g > g_cap */
    int64_t reflected;    /* cumulative electrons reflected at a wall */
    int64_t n_pairs;      /* cumulative binary Coulomb collisions */
} pic1d_moments_t;

/*
 * Size query: bytes of device workspace pic1d_create needs for this config.  HOST pointers.
 */
int pic1d_workspace_bytes(const pic1d_config_t* cfg, size_t* bytes_out);

/*
 * Create a handle.  cfg: HOST pointer, copied.  workspace: DEVICE memory, 256-byte aligned, at least
 * pic1d_workspace_bytes() long, owned by the caller and kept alive until pic1d_destroy.
 * cuda_stream: the caller's cudaStream_t (NULL = default stream).  *out receives the handle.
 * (Problem statement L33-41; data structure L63-67.)
 */
int pic1d_create(const pic1d_config_t* cfg, void* workspace, size_t workspace_bytes, void* cuda_stream,
                 pic1d_t** out);

/*
 * Load species `species` (L63): n particles, x in [0, N_c) grid-cell units, velocities in cells/step
 * taken as v(-dt/2) (leapfrog, L150).  Arrays are HOST (on_device = 0) or DEVICE (on_device = 1)
 * fp32, copied; the caller keeps ownership.  When the last species has been loaded the library
 * fine-sorts, deposits and solves, so rho/phi/E are valid for step 0 and the step counter is 0.
 * n > capacity -> PIC1D_ERR_CAPACITY; x outside [0, N_c) -> PIC1D_ERR_ARG (checked on the device).
 */
int pic1d_load_particles(pic1d_t* h, int species, int64_t n, const float* x, const float* vx,
                         const float* vy, const float* vz, int on_device);

/*
 * Enqueue n_steps full PIC/MCC cycles (Fig. 1, L35-41) on the stream.  Asynchronous: no host
 * synchronisation, no host round trip of rho or E (contrast L144).  Errors raised inside the
 * kernels are sticky and surface on the next synchronising call.  Pairs of steps are replayed from a
 * CUDA graph captured on first use (the step index and every particle count are device-resident).
 */
int pic1d_step(pic1d_t* h, int n_steps);

/*
 * Copy net charge density rho (raw linear-weighting sums, no wall-node doubling), potential phi and
 * field E (Eq. 1-2), fp64, n_nodes values each, to HOST (on_device = 0; synchronises) or
 * DEVICE (on_device = 1; enqueued) buffers.  Any pointer may be NULL.  Returns the sticky error.
 */
int pic1d_get_rho_phi_E(pic1d_t* h, double* rho, double* phi, double* E, int n_nodes, int on_device);

/*
 * Moments of species `species` (synchronises).  out: HOST.  density: optional HOST buffer of
 * n_density = n_nodes doubles receiving rho_s of the last deposit (number density per node).
 * eedf: optional HOST buffer of n_bins int64 receiving the histogram of E = c_eV |v|^2 on [0, E_max).
 */
int pic1d_moments(pic1d_t* h, int species, pic1d_moments_t* out, double* density, int n_density,
                  int64_t* eedf, int n_bins, double E_max);

/* Free the host-side handle.  The workspace stays the caller's. */
int pic1d_destroy(pic1d_t* h);

/* ---- helpers outside the six-call contract ------------------------------------------------- */
int pic1d_abi_version(void); /* PIC1D_ABI_VERSION of the library that is loaded */
int pic1d_n_nodes(const pic1d_t* h);
int pic1d_n_sort_cells(const pic1d_t* h);
uint32_t pic1d_step_index(const pic1d_t* h);
const char* pic1d_last_cuda_error(const pic1d_t* h);
/* number of kernel launches enqueued by this handle since creation */
int64_t pic1d_launch_count(const pic1d_t* h);
/* number of CUDA-graph replays (two steps each) pic1d_step has launched since creation; -1 once a capture or an
 * instantiation has failed (e.g. on the legacy default stream): the handle then launches every kernel itself for
 * good, with identical results.  0 with PIC1D_FLAG_NO_GRAPH. */
int64_t pic1d_graph_launch_count(const pic1d_t* h);

/* Per-kernel timing (host API, synchronises): runs ONE step with CUDA events between the kernels
 * and writes up to max_kernels entries of (name, milliseconds).  Returns the number of entries. */
typedef struct pic1d_kernel_time {
    char name[48];
    float ms;
    int32_t species; /* -1 = not species specific */
} pic1d_kernel_time_t;
int pic1d_step_timed(pic1d_t* h, pic1d_kernel_time_t* out, int max_kernels);

/* Debug access for the parity harness (synchronises).  `what` selects the array; *count_out gets
 * the element count; dst (HOST) must hold `bytes` >= count * element size. */
enum pic1d_debug_what {
    PIC1D_DBG_X = 0,   /* float[N_s]  */
    PIC1D_DBG_VX = 1,
    PIC1D_DBG_VY = 2,
    PIC1D_DBG_VZ = 3,
    PIC1D_DBG_KEYS = 4,    /* int32 per pre-sort slot of the last step, -1 = absorbed (needs CAPTURE) */
    PIC1D_DBG_OFFSETS = 5, /* int32[N_sc + 1] */
    PIC1D_DBG_MASK = 6,    /* uint8 per sorted slot: MCC event of the last step (needs CAPTURE) */
    PIC1D_DBG_E32 = 7,     /* float[n_nodes]: the field the next push will gather */
    PIC1D_DBG_RHO_S = 8,   /* double[n_nodes]: rho_s of the last deposit */
    PIC1D_DBG_TILE_W = 9,  /* int32 per tile of the last sort: width (sort cells) of the tile's key window */
    PIC1D_DBG_PARTNER = 10 /* int32 per sorted slot: partner of the last step's binary collisions, -1 = none (needs CAPTURE) */
};
int pic1d_debug_count(pic1d_t* h, int what, int species, int64_t* count_out);
int pic1d_debug_get(pic1d_t* h, int what, int species, void* dst, size_t bytes);
/* Overwrite the fp32 field the next push gathers (so a single-step parity test can start from an
 * identical state, R17).  E32: HOST, n_nodes floats. */
int pic1d_debug_set_E32(pic1d_t* h, const float* E32, int n_nodes);

/* Overwrite the live particles of a species IN PLACE, keeping their order: slots [0, n_sorted) are taken as
 * the sorted part, [n_sorted, n) as the birth tail; nothing is sorted, deposited or solved.  step >= 0 also sets
 * the index of the next step.  The parity harness uses it to start EVERY compared step from the oracle's exact
 * state (velocities of collided particles otherwise differ in the last bits: libm vs CUDA sin / cos / log), so
 * that the single-step bars of north_star (x bit-exact, rho 1e-9) apply to every step.  HOST arrays, copied. */
int pic1d_debug_set_state(pic1d_t* h, int species, int64_t n, int64_t n_sorted, const float* x, const float* vx,
                          const float* vy, const float* vz, int64_t step);

#ifdef __cplusplus
}
#endif
#endif /* PIC1D_H_ */
