/*
 * pic1d_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded CPU statement of one 1D3V electrostatic PIC/MCC
 * cycle with per-cell fine sorting, written from the paper
 *   Mertmann et al., "Fine-sorting One-dimensional Particle-In-Cell Algorithm with
 *   Monte-Carlo Collisions on a Graphics Processing Unit"
 * step by step in the paper's order and notation.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or helper with the CUDA path under paper_1104_3998_b200/csrc/.
 *
 * Compile:  gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -shared -fPIC
 * (-ffp-contract=off: every fp32 operation below is exactly the IEEE operation that is
 *  written; fmaf() appears only where the step definition says "fma".)
 *
 * Cycle (Fig. 1), entered at the pusher with E^n valid (R2):
 *   1 gather + leapfrog push      L35, L150-156, Eq. 3-4 (L119-122), L152-154
 *   2 wall absorption, secondary-electron injection, compaction           L41
 *   3 fine sort: key = sort cell, counting sort, stable       L63-67, L160-192
 *   4 charge deposition, linear weighting        L35, L128-138, Fig. 4 (L99)
 *   5 Poisson (Thomas) + E                 Eq. 1-2 (L113-117), L142-146
 *   6 modified null-collision Monte-Carlo collisions   L196-209, Eq. 6 (L200)
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"), per function:
 *   philox4x32_10 : cuRAND host generator CURAND_RNG_PHILOX4_32_10 (independent code),
 *                   bijectivity on two 2^16 sub-cubes of the counter space, uniformity
 *   u01           : range / mean / chi^2 of U(r); Eq. 6 candidate rate
 *   push (step 1) : constant-field and linear-field closed forms (leapfrog), linear gather
 *   boundary, SEE : bookkeeping, ties at the walls, order, SEE binomial + Rayleigh moments;
 *                   periodic wrap incl. the |v| > N_c / non-finite clamp (R21)
 *   sort_species  : permutation, brute-force offsets, stability, numpy stable argsort
 *   deposit       : sum(rho_s) == N_s exactly, single particle, brute-force hat sum, wrap
 *   thomas_dirichlet, field_solve (the function the cycle runs; oracle_solve_field calls it):
 *                   uniform / sinusoidal / Laplace / single-sheet closed forms incl. both
 *                   wall nodes, Gauss's law over the gap, dense numpy solve; the uniform
 *                   plasma through load -> sort -> deposit -> field_solve of the full Oracle
 *   mcc           : null-collision statistics (Eq. 6); beam fractions against values built
 *                   from the physical inputs (n_g, sigma_k(E), v(E), dt); kinematic
 *                   invariants (energy bookkeeping, isotropy, Maxwellian moments)
 *   oracle_moments: numpy sums and numpy.histogram on the arrays debug_get returns;
 *                   Maxwellian <v^2>, <v^4>
 *   whole loop    : cold plasma oscillation frequency (config 1), momentum conservation
 *   binary_collide (f3), reflect (f4), gapped sort (f2): see their own headers below
 *   long RF discharge physics (configs 2-4): parity unpinned beyond bookkeeping.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_MAX_SPECIES 2

/* Philox stream ids (R12) */
#define STREAM_NULL 0u /* + species index */
#define STREAM_COLL 2u /* + species index */
#define STREAM_SEE 4u
#define STREAM_REFL 5u /* electron reflection at the walls (f4) */
#define STREAM_COUL 6u /* + species index: binary Coulomb collisions inside sort cells (f3) */

typedef struct {
    double kappa;     /* signed push constant kappa_s, Eq. 3 (L119) */
    double c_eV;      /* eV per (cell/step)^2 */
    double P0;        /* null-collision probability, Eq. 6 (L200) */
    double inv_g_cap; /* 1 / g_cap [steps/cell] */
    int64_t capacity; /* slots */
    int32_t charge_sign;
    int32_t mcc_kind; /* 0 none, 1 electron set, 2 ion charge exchange */
} orc_species_cfg;

typedef struct {
    uint32_t struct_size;
    int32_t n_cells;   /* N_c grid cells */
    int32_t bc;        /* 0 bounded (absorbing walls), 1 periodic */
    int32_t n_species; /* 1 or 2; species 0 = electrons, 1 = ions */
    orc_species_cfg sp[ORC_MAX_SPECIES];
    double background_rho; /* periodic neutraliser */
    double sort_inv_ratio; /* 1/r, power of two */
    double V0_norm, omega_dt;
    double see_gamma, see_vth;
    double r_el, r_exc, r_ion; /* sigma_k0 / sigma_cap */
    double E_exc, E_ion;       /* eV */
    double gas_vth_ion;        /* cells/step */
    double mass_ratio;         /* m_e / M */
    uint64_t seed;
    uint32_t flags;
    uint32_t pad_;
    double e_reflect; /* probability that an electron reaching a wall is reflected (L41; R22) */
    double coul_A[ORC_MAX_SPECIES]; /* binary collisions in sort cells (L69): <tan^2(theta/2)> =
                                       coul_A n_cell / u^3, u in cells/step; 0 = off (R23) */
} orc_config;

typedef struct {
    int64_t count, n_sorted;
    double sum_vx, sum_vy, sum_vz, sum_v2, sum_v4;
    int64_t absorbed_left, absorbed_right;
    int64_t injected;     /* secondary electrons injected into this species */
    int64_t n_candidates; /* passed the null test */
    int64_t n_events[4];  /* [0] null, [1] elastic / CX, [2] excitation, [3] ionisation */
    int64_t births;       /* ionisation births appended to this species */
    int64_t dropped;      /* births / injections dropped for lack of capacity */
    int64_t over_cap;     /* candidates with g > g_cap */
    int64_t reflected;    /* electrons reflected at a wall (f4) */
    int64_t n_pairs;      /* binary collisions performed (f3) */
} orc_moments;

typedef struct {
    float *x, *vx, *vy, *vz;     /* state, capacity slots */
    float *tx, *tvx, *tvy, *tvz; /* sort destination */
    int32_t* src_key;            /* key per pre-sort slot, -1 = absorbed (debug) */
    uint8_t* mask;               /* MCC event per sorted slot */
    int32_t* offsets;            /* n_sc + 1 */
    int32_t* partner;            /* f3: partner slot of each sorted slot in the last step, -1 = unpaired */
    double* rho_s;               /* nodes (+1 scratch for periodic wrap) */
    int64_t n, n_sorted, n_src;
    orc_moments m; /* cumulative counters live here */
} orc_species;

typedef struct {
    orc_config cfg;
    int nodes, n_sc;
    float inv_r;
    orc_species sp[ORC_MAX_SPECIES];
    double *rho, *phi, *E, *tmp;
    float* E32;
    uint32_t step;
    int loaded_mask;
    int error;
    /* absorbed-ion list of the current step */
    int64_t* abs_slot;
    uint8_t* abs_wall;
    int64_t n_abs, abs_cap;
} orc_t;

/* ------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): counter-based generator that
 * replaces the paper's per-thread xorshift (L205) -- DESIGN.md R12.
 * ---------------------------------------------------------------------------------- */
static void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                          uint32_t k1, uint32_t out[4]) {
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void oracle_philox(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                   uint32_t out[4]) {
    philox4x32_10(c0, c1, c2, c3, (uint32_t)seed, (uint32_t)(seed >> 32), out);
}

/* U(r) = (r >> 8) * 2^-24 in [0,1), exact in fp32 */
static float u01(uint32_t r) { return (float)(r >> 8) * 0x1p-24f; }

static void philox_u(const orc_t* o, uint32_t c0, uint32_t stream, uint32_t blk, float u[4]) {
    uint32_t w[4];
    philox4x32_10(c0, o->step, stream, blk, (uint32_t)o->cfg.seed,
                  (uint32_t)(o->cfg.seed >> 32), w);
    for (int k = 0; k < 4; ++k) u[k] = u01(w[k]);
}

/* ------------------------------------------------------------------------------------ */
static void free_species(orc_species* s) {
    free(s->x); free(s->vx); free(s->vy); free(s->vz);
    free(s->tx); free(s->tvx); free(s->tvy); free(s->tvz);
    free(s->src_key); free(s->mask); free(s->offsets); free(s->rho_s); free(s->partner);
    memset(s, 0, sizeof(*s));
}

int oracle_destroy(orc_t* o) {
    if (!o) return 0;
    for (int s = 0; s < ORC_MAX_SPECIES; ++s) free_species(&o->sp[s]);
    free(o->rho); free(o->phi); free(o->E); free(o->tmp); free(o->E32);
    free(o->abs_slot); free(o->abs_wall);
    free(o);
    return 0;
}

int oracle_create(const orc_config* cfg, orc_t** out) {
    if (!cfg || !out || cfg->struct_size != sizeof(orc_config)) return -1;
    if (cfg->n_cells < 2 || cfg->n_species < 1 || cfg->n_species > ORC_MAX_SPECIES) return -1;
    if (!(cfg->sort_inv_ratio > 0.0)) return -1;
    orc_t* o = (orc_t*)calloc(1, sizeof(orc_t));
    if (!o) return -1;
    o->cfg = *cfg;
    o->nodes = cfg->bc == 1 ? cfg->n_cells : cfg->n_cells + 1;
    o->inv_r = (float)cfg->sort_inv_ratio;
    o->n_sc = (int)ceil((double)cfg->n_cells * cfg->sort_inv_ratio); /* N_sc, R9 */
    for (int s = 0; s < cfg->n_species; ++s) {
        orc_species* p = &o->sp[s];
        size_t cap = (size_t)cfg->sp[s].capacity;
        p->x = malloc(cap * 4); p->vx = malloc(cap * 4); p->vy = malloc(cap * 4); p->vz = malloc(cap * 4);
        p->tx = malloc(cap * 4); p->tvx = malloc(cap * 4); p->tvy = malloc(cap * 4); p->tvz = malloc(cap * 4);
        p->src_key = malloc(cap * 4);
        p->mask = calloc(cap, 1);
        p->offsets = calloc((size_t)o->n_sc + 1, 4);
        p->rho_s = calloc((size_t)o->nodes + 1, 8);
        p->partner = malloc(cap * 4);
    }
    o->rho = calloc((size_t)o->nodes + 1, 8);
    o->phi = calloc((size_t)o->nodes + 1, 8);
    o->E = calloc((size_t)o->nodes + 1, 8);
    o->tmp = calloc((size_t)o->nodes + 1, 8);
    o->E32 = calloc((size_t)o->nodes + 1, 4);
    o->abs_cap = cfg->n_species > 1 ? cfg->sp[1].capacity : 1;
    o->abs_slot = malloc((size_t)o->abs_cap * 8);
    o->abs_wall = malloc((size_t)o->abs_cap);
    *out = o;
    return 0;
}

/* ---- step 3: fine sort (L63-67, L160-192): key = (int)(x * inv_r); histogram; exclusive
 * scan -> offsets; stable scatter in input order.  Plain definition: stable sort by key,
 * offsets[k] = #{p : key_p < k}. */
static void sort_species(orc_t* o, int s) {
    orc_species* p = &o->sp[s];
    int n_sc = o->n_sc;
    int64_t n = p->n;
    int32_t* cur = (int32_t*)calloc((size_t)n_sc + 1, 4);
    for (int64_t i = 0; i < n; ++i) {
        int key = (int)(p->x[i] * o->inv_r);
        cur[key + 1]++;
    }
    for (int k = 0; k < n_sc; ++k) cur[k + 1] += cur[k];
    memcpy(p->offsets, cur, ((size_t)n_sc + 1) * 4);
    for (int64_t i = 0; i < n; ++i) {
        int key = (int)(p->x[i] * o->inv_r);
        int32_t d = cur[key]++;
        p->tx[d] = p->x[i]; p->tvx[d] = p->vx[i]; p->tvy[d] = p->vy[i]; p->tvz[d] = p->vz[i];
    }
    free(cur);
    float* t;
    t = p->x; p->x = p->tx; p->tx = t;
    t = p->vx; p->vx = p->tvx; p->tvx = t;
    t = p->vy; p->vy = p->tvy; p->tvy = t;
    t = p->vz; p->vz = p->tvz; p->tvz = t;
    p->n_sorted = n;
}

/* ---- step 4: charge deposition, linear weighting onto the two neighbouring nodes
 * (L35, L128-138, Fig. 4).  fp64 accumulation; rho_s is the RAW sum (R8). */
static void deposit(orc_t* o) {
    int Nc = o->cfg.n_cells;
    for (int s = 0; s < o->cfg.n_species; ++s) {
        orc_species* p = &o->sp[s];
        memset(p->rho_s, 0, ((size_t)o->nodes + 1) * 8);
        for (int64_t i = 0; i < p->n_sorted; ++i) {
            float x = p->x[i];
            int j = (int)x;
            float f = x - (float)j;
            double w1 = (double)f, w0 = 1.0 - w1;
            int j1 = j + 1;
            if (o->cfg.bc == 1 && j1 == Nc) j1 = 0; /* node N_c == node 0 */
            p->rho_s[j] += w0;
            p->rho_s[j1] += w1;
        }
    }
    for (int j = 0; j < o->nodes; ++j) {
        double r = o->cfg.background_rho;
        for (int s = 0; s < o->cfg.n_species; ++s)
            r += (double)o->cfg.sp[s].charge_sign * o->sp[s].rho_s[j];
        o->rho[j] = r;
    }
}

/* Thomas algorithm (L142, ref. [16]) for  phi[j-1] - 2 phi[j] + phi[j+1] = -rhs[j],
 * j = 1..n-1, phi[0] and phi[n] given.  cp = scratch of n+1 doubles. */
static void thomas_dirichlet(int n, const double* rhs, double* phi, double* cp) {
    /* written as  -phi[j-1] + 2 phi[j] - phi[j+1] = rhs[j]  (a=-1, b=2, c=-1) */
    if (n < 2) return;
    double* dp = phi; /* reuse phi[1..n-1] for the modified right-hand side */
    double b = 2.0;
    cp[1] = -1.0 / b;
    dp[1] = (rhs[1] + phi[0]) / b;
    for (int j = 2; j <= n - 1; ++j) {
        double d = rhs[j];
        if (j == n - 1) d += phi[n];
        double m = b + cp[j - 1]; /* b - a*cp[j-1], a = -1 */
        cp[j] = -1.0 / m;
        dp[j] = (d + dp[j - 1]) / m;
    }
    if (n - 1 == 1) dp[1] = (rhs[1] + phi[0] + phi[n]) / b;
    for (int j = n - 2; j >= 1; --j) dp[j] = dp[j] - cp[j] * dp[j + 1];
}

/* ---- step 5: Poisson + E (Eq. 1-2) for the wall potentials phi_0 = phi0 and
 * phi_{N_c} = phiN (bounded; ignored for periodic runs). */
static void field_solve(orc_t* o, double phi0, double phiN) {
    int Nc = o->cfg.n_cells;
    double *rho = o->rho, *phi = o->phi, *E = o->E;
    if (o->cfg.bc == 0) {
        phi[0] = phi0;
        phi[Nc] = phiN;
        thomas_dirichlet(Nc, rho, phi, o->tmp);
        for (int j = 1; j < Nc; ++j) E[j] = (phi[j - 1] - phi[j + 1]) / 2.0;
        /* half-cell Gauss law with the RAW wall-node sums (R7) */
        E[0] = (phi[0] - phi[1]) - rho[0];
        E[Nc] = (phi[Nc - 1] - phi[Nc]) + rho[Nc];
    } else {
        double mean = 0.0;
        for (int j = 0; j < Nc; ++j) mean += rho[j];
        mean /= (double)Nc;
        double* r = (double*)calloc((size_t)Nc + 1, 8);
        for (int j = 0; j < Nc; ++j) r[j] = rho[j] - mean;
        phi[0] = 0.0;
        phi[Nc] = 0.0; /* node N_c == node 0 */
        thomas_dirichlet(Nc, r, phi, o->tmp);
        free(r);
        for (int j = 0; j < Nc; ++j) {
            int jm = j == 0 ? Nc - 1 : j - 1, jp = j == Nc - 1 ? 0 : j + 1;
            E[j] = (phi[jm] - phi[jp]) / 2.0;
        }
        double pm = 0.0;
        for (int j = 0; j < Nc; ++j) pm += phi[j];
        pm /= (double)Nc;
        for (int j = 0; j < Nc; ++j) phi[j] -= pm;
    }
    for (int j = 0; j < o->nodes; ++j) o->E32[j] = (float)E[j];
}

/* wall potentials at time t_n = n_time * dt (R6): node 0 driven, node N_c grounded */
static void field_solve_at(orc_t* o, uint32_t n_time) {
    field_solve(o, o->cfg.V0_norm * sin(o->cfg.omega_dt * (double)n_time), 0.0);
}

/* isotropic unit vector from two uniforms (R14) */
static void iso_dir(float ua, float ub, float n[3]) {
    float ct = 1.0f - 2.0f * ua;
    float st = sqrtf(fmaxf(0.0f, 1.0f - ct * ct));
    float ph = 6.2831855f * ub;
    n[0] = ct;
    n[1] = st * cosf(ph);
    n[2] = st * sinf(ph);
}

/* one standard normal pair member: sqrt(-2 ln(1-u)) * cos/sin(2 pi w) (Box-Muller) */
static float bm_r(float u) { return sqrtf(-2.0f * logf(1.0f - u)); }

/* ---- step 6: modified null-collision MCC (L196-209, Eq. 6): EVERY particle draws p;
 * p < P0 enters the standard null-collision selection.  One particle = one id = its
 * sorted slot.  Ionisation products are born at the parent's position (L203) and are
 * appended to the tails in ascending parent-slot order. */
static void mcc(orc_t* o) {
    const orc_config* c = &o->cfg;
    for (int s = 0; s < c->n_species; ++s) {
        orc_species* p = &o->sp[s];
        int kind = c->sp[s].mcc_kind;
        if (kind == 0) continue;
        float P0 = (float)c->sp[s].P0;
        float inv_g_cap = (float)c->sp[s].inv_g_cap;
        float c_eV = (float)c->sp[s].c_eV;
        float r_el = (float)c->r_el, r_exc = (float)c->r_exc, r_ion = (float)c->r_ion;
        float E_exc = (float)c->E_exc, E_ion = (float)c->E_ion;
        float two_mr = (float)(2.0 * c->mass_ratio);
        float gvt = (float)c->gas_vth_ion;
        int64_t ns = p->n_sorted;
        int64_t births = 0;
        for (int64_t i = 0; i < ns; ++i) {
            p->mask[i] = 0;
            float u4[4];
            philox_u(o, (uint32_t)(i >> 2), STREAM_NULL + (uint32_t)s, 0u, u4);
            float u0 = u4[i & 3];
            if (!(u0 < P0)) continue;
            p->m.n_candidates++;
            float b0[4];
            philox_u(o, (uint32_t)i, STREAM_COLL + (uint32_t)s, 0u, b0);
            float u_type = b0[0], u_a = b0[1], u_b = b0[2], u_c = b0[3];
            float vx = p->vx[i], vy = p->vy[i], vz = p->vz[i];
            float g2 = (vx * vx + vy * vy) + vz * vz;
            float g = sqrtf(g2);
            float a = g * inv_g_cap;
            if (a > 1.0f) p->m.over_cap++;
            if (kind == 1) {
                float En = c_eV * g2;
                float P_el = a * r_el;
                float P_exc = En > E_exc ? (a * r_exc) * (1.0f - E_exc / En) : 0.0f;
                float P_ion = En > E_ion ? (a * r_ion) * (1.0f - E_ion / En) : 0.0f;
                float t1 = P_el, t2 = t1 + P_exc, t3 = t2 + P_ion;
                int ev = u_type < t1 ? 1 : (u_type < t2 ? 2 : (u_type < t3 ? 3 : 0));
                p->mask[i] = (uint8_t)ev;
                p->m.n_events[ev]++;
                if (ev == 0) continue;
                float n[3];
                iso_dir(u_a, u_b, n);
                float gp;
                if (ev == 1) {
                    float cchi = ((n[0] * vx + n[1] * vy) + n[2] * vz) / g;
                    gp = g * sqrtf(1.0f - two_mr * (1.0f - cchi));
                } else if (ev == 2) {
                    gp = sqrtf((En - E_exc) / c_eV);
                } else {
                    gp = sqrtf(((En - E_ion) * 0.5f) / c_eV);
                }
                p->vx[i] = gp * n[0]; p->vy[i] = gp * n[1]; p->vz[i] = gp * n[2];
                if (ev == 3) {
                    /* pair: second electron, same speed, independent direction; Ar+ at the
                     * same x with Maxwellian gas velocity */
                    orc_species* pe = &o->sp[0];
                    orc_species* pi = c->n_species > 1 ? &o->sp[1] : NULL;
                    int ok = pe->n < c->sp[0].capacity && (!pi || pi->n < c->sp[1].capacity);
                    if (!ok) {
                        pe->m.dropped++;
                        if (pi) pi->m.dropped++;
                        o->error = -2;
                        continue;
                    }
                    float b1[4], b2[4];
                    philox_u(o, (uint32_t)i, STREAM_COLL + (uint32_t)s, 1u, b1);
                    philox_u(o, (uint32_t)i, STREAM_COLL + (uint32_t)s, 2u, b2);
                    float n2[3];
                    iso_dir(u_c, b1[0], n2);
                    int64_t de = pe->n++;
                    pe->x[de] = p->x[i];
                    pe->vx[de] = gp * n2[0]; pe->vy[de] = gp * n2[1]; pe->vz[de] = gp * n2[2];
                    pe->m.births++;
                    if (pi) {
                        float r12 = bm_r(b1[1]), ph12 = 6.2831855f * b1[2];
                        float r3 = bm_r(b1[3]), ph3 = 6.2831855f * b2[0];
                        int64_t di = pi->n++;
                        pi->x[di] = p->x[i];
                        pi->vx[di] = gvt * (r12 * cosf(ph12));
                        pi->vy[di] = gvt * (r12 * sinf(ph12));
                        pi->vz[di] = gvt * (r3 * cosf(ph3));
                        pi->m.births++;
                    }
                    births++;
                }
            } else { /* kind == 2: ion charge exchange with the cold background gas */
                float P_cx = fminf(1.0f, a);
                int ev = u_type < P_cx ? 1 : 0;
                p->mask[i] = (uint8_t)ev;
                p->m.n_events[ev]++;
                if (ev == 0) continue;
                float b1[4];
                philox_u(o, (uint32_t)i, STREAM_COLL + (uint32_t)s, 1u, b1);
                float r12 = bm_r(u_a), ph12 = 6.2831855f * u_b;
                float r3 = bm_r(u_c), ph3 = 6.2831855f * b1[0];
                p->vx[i] = gvt * (r12 * cosf(ph12));
                p->vy[i] = gvt * (r12 * sinf(ph12));
                p->vz[i] = gvt * (r3 * cosf(ph3));
            }
        }
        (void)births;
    }
}

/* ---- step 6b (f3): binary Coulomb collisions inside sort cells (L69, L75, L221, L259: the reason
 * the paper sorts finely; it does not implement them).  Takizuka & Abe's binary collision model
 * (J. Comput. Phys. 25 (1977) 205), like particles of one species (equal mass, equal weight):
 * the n particles of a sort cell are paired; a pair with relative velocity u = v_a - v_b is
 * scattered by the angle theta, tan(theta/2) = delta ~ N(0, <delta^2>),
 * <delta^2> = coul_A n / u^3 (coul_A = q^4 w lnLambda dt / (8 pi eps0^2 m_r^2 V_cell), m_r = m/2,
 * in normalised units, computed by the caller), azimuth phi uniform; u is rotated, each partner takes
 * half of the change: momentum and energy of the pair are conserved.
 * Pairing (R23; the paper gives none, Takizuka-Abe pair at random): a keyed pseudo-random
 * permutation pi of the cell's sorted slots 0 .. n-1; pairs are (pi(2m), pi(2m+1)); for odd n slot pi(n-1)
 * sits out (Takizuka-Abe's three-particle rule for odd n is NOT used).  pi is a 4-round balanced Feistel
 * network on 2h bits, h the smallest integer with 4^h >= n, keyed by the four words of
 * philox(cell, step, COUL + s, 0), made a permutation of [0, n) by cycle walking (apply again while the value
 * is >= n: a cycle of a permutation of [0, 4^h) that starts below n comes back below n).  Any pairing of the
 * cell can come out, unlike the single-stride pairs of an affine map (a m + b) mod n. */
static uint32_t coul_mix(uint32_t z) { /* round function: an integer hash, the low h bits are used */
    z *= 0x9E3779B1u; z ^= z >> 15; z *= 0x85EBCA77u; z ^= z >> 13;
    return z;
}

static uint32_t coul_perm(uint32_t m, uint32_t n, uint32_t h, const uint32_t w[4]) {
    const uint32_t mask = (1u << h) - 1u;
    uint32_t x = m;
    do {
        uint32_t L = x >> h, R = x & mask;
        for (int r = 0; r < 4; ++r) {
            uint32_t t = L ^ (coul_mix(R ^ w[r]) & mask);
            L = R; R = t;
        }
        x = (L << h) | R;
    } while (x >= n);
    return x;
}

static void coulomb(orc_t* o) {
    const orc_config* c = &o->cfg;
    for (int s = 0; s < c->n_species; ++s) {
        orc_species* p = &o->sp[s];
        float A = (float)c->coul_A[s];
        for (int64_t i = 0; i < p->n_sorted; ++i) p->partner[i] = -1;
        if (!(A > 0.0f)) continue;
        for (int k = 0; k < o->n_sc; ++k) {
            uint32_t off = (uint32_t)p->offsets[k], n = (uint32_t)(p->offsets[k + 1] - p->offsets[k]);
            if (n < 2) continue;
            uint32_t w[4];
            philox4x32_10((uint32_t)k, o->step, STREAM_COUL + (uint32_t)s, 0u, (uint32_t)c->seed,
                          (uint32_t)(c->seed >> 32), w);
            uint32_t h = 1;
            while ((1ull << (2 * h)) < n) ++h; /* 4^h >= n */
            float fn = (float)n;
            for (uint32_t m = 0; m + 1 < n; m += 2) {
                uint32_t ia = off + coul_perm(m, n, h, w);
                uint32_t ib = off + coul_perm(m + 1, n, h, w);
                p->partner[ia] = (int32_t)ib; p->partner[ib] = (int32_t)ia;
                p->m.n_pairs++;
                float u4[4];
                philox_u(o, ia, STREAM_COUL + (uint32_t)s, 1u, u4); /* keyed on the pair's first slot */
                float ux = p->vx[ia] - p->vx[ib], uy = p->vy[ia] - p->vy[ib], uz = p->vz[ia] - p->vz[ib];
                float up2 = ux * ux + uy * uy;
                float u2 = up2 + uz * uz;
                if (!(u2 > 0.0f)) continue;
                float uu = sqrtf(u2), up = sqrtf(up2);
                float var = (A * fn) / (u2 * uu);
                float delta = sqrtf(var) * (bm_r(u4[0]) * cosf(6.2831855f * u4[1]));
                float d2 = delta * delta;
                float sint = (2.0f * delta) / (1.0f + d2);
                float omc = (2.0f * d2) / (1.0f + d2); /* 1 - cos(theta) */
                float ph = 6.2831855f * u4[2];
                float cp = cosf(ph), sp_ = sinf(ph);
                float dux, duy, duz;
                if (up > 0.0f) {
                    dux = ((ux / up) * uz) * (sint * cp) - ((uy / up) * uu) * (sint * sp_) - ux * omc;
                    duy = ((uy / up) * uz) * (sint * cp) + ((ux / up) * uu) * (sint * sp_) - uy * omc;
                    duz = -(up * (sint * cp)) - uz * omc;
                } else {
                    dux = uu * (sint * cp); duy = uu * (sint * sp_); duz = -(uz * omc);
                }
                p->vx[ia] += 0.5f * dux; p->vy[ia] += 0.5f * duy; p->vz[ia] += 0.5f * duz;
                p->vx[ib] -= 0.5f * dux; p->vy[ib] -= 0.5f * duy; p->vz[ib] -= 0.5f * duz;
            }
        }
    }
}

/* ---- step 1 for ONE particle: gather (linear weighting, L35) + leapfrog push (L150-156):
 *   v(t+1/2) = v(t-1/2) + kappa E(x(t));   x(t+1) = x(t) + v(t+1/2)   (L152-154) */
static void gather_push(const float* E32, float kappa, int Nc, int bc, float* px, float* pvx) {
    float x = *px;
    int j = (int)x; /* "single type casting operation", L87 */
    float f = x - (float)j;
    int j1 = j + 1;
    if (bc == 1 && j1 == Nc) j1 = 0;
    float Ep = fmaf(f, E32[j1] - E32[j], E32[j]);
    float v = fmaf(kappa, Ep, *pvx);
    *pvx = v;
    *px = x + v;
}

/* ---- one full step n -> n+1 ------------------------------------------------------ */
static void step_once(orc_t* o) {
    const orc_config* c = &o->cfg;
    int Nc = c->n_cells;
    float fNc = (float)Nc;
    /* 1. gather + push (L35, L150-156):  v(t+1/2) = v(t-1/2) + kappa E(x(t));
     *    x(t+1) = x(t) + v(t+1/2)   (L152-154) */
    for (int s = 0; s < c->n_species; ++s) {
        orc_species* p = &o->sp[s];
        float kappa = (float)c->sp[s].kappa;
        for (int64_t i = 0; i < p->n; ++i) gather_push(o->E32, kappa, Nc, c->bc, &p->x[i], &p->vx[i]);
    }
    /* 2. boundary (L41): electrons first, then ions */
    o->n_abs = 0;
    int64_t n_before[ORC_MAX_SPECIES] = {0, 0};
    for (int s = 0; s < c->n_species; ++s) {
        orc_species* p = &o->sp[s];
        n_before[s] = p->n;
        int64_t w = 0;
        for (int64_t i = 0; i < p->n; ++i) {
            float x = p->x[i];
            if (c->bc == 1) {
                if (x < 0.0f) x += fNc;
                if (x >= fNc) x -= fNc;
                /* rounding of -tiny + N_c, |v| > N_c, or non-finite: back to x = 0 */
                if (!(x >= 0.0f && x < fNc)) x = 0.0f;
            } else if (!(x >= 0.0f && x < fNc)) {
                /* f4, electron reflection (L41: "If ... electron reflection are featured, electrons are
                 * inserted at the boundaries"; R22): with probability e_reflect the electron is
                 * put back at the mirror position with vx reversed, and stays where it was in the order */
                if (s == 0 && c->e_reflect > 0.0 && x == x) {
                    float u[4];
                    philox_u(o, (uint32_t)i, STREAM_REFL, 0u, u);
                    if (u[0] < (float)c->e_reflect) {
                        float xr = x < 0.0f ? -x : (2.0f * fNc) - x;
                        if (xr >= 0.0f && xr < fNc) {
                            p->m.reflected++;
                            p->vx[i] = -p->vx[i];
                            p->src_key[i] = (int)(xr * o->inv_r);
                            p->x[w] = xr; p->vx[w] = p->vx[i]; p->vy[w] = p->vy[i]; p->vz[w] = p->vz[i];
                            ++w;
                            continue;
                        }
                    }
                }
                if (x != x) o->error = -4;
                if (x < 0.0f) p->m.absorbed_left++; else p->m.absorbed_right++;
                p->src_key[i] = -1;
                if (s == 1 && c->sp[s].charge_sign > 0 && c->see_gamma > 0.0 &&
                    o->n_abs < o->abs_cap) {
                    o->abs_slot[o->n_abs] = i;
                    o->abs_wall[o->n_abs] = x < 0.0f ? 0 : 1;
                    o->n_abs++;
                }
                continue;
            }
            p->src_key[i] = (int)(x * o->inv_r);
            p->x[w] = x; p->vx[w] = p->vx[i]; p->vy[w] = p->vy[i]; p->vz[w] = p->vz[i];
            ++w;
        }
        p->n = w;
    }
    /* secondary-electron emission at ion impact (L41), ascending ion-slot order */
    if (o->n_abs > 0) {
        orc_species* pe = &o->sp[0];
        float gamma = (float)c->see_gamma, svt = (float)c->see_vth;
        int64_t n_inj = 0;
        for (int64_t a = 0; a < o->n_abs; ++a) {
            uint32_t i = (uint32_t)o->abs_slot[a];
            float u[4], u2[4];
            philox_u(o, i, STREAM_SEE, 0u, u);
            if (!(u[0] < gamma)) continue;
            /* capacity counts the slots in use at the start of the step plus injections */
            if (n_before[0] + n_inj >= c->sp[0].capacity) {
                pe->m.dropped++;
                o->error = -2;
                continue;
            }
            philox_u(o, i, STREAM_SEE, 1u, u2);
            float x, sgn;
            if (o->abs_wall[a] == 0) {
                x = u[1];
                sgn = 1.0f;
            } else {
                x = fminf(fNc - (1.0f - u[1]), nextafterf(fNc, 0.0f));
                sgn = -1.0f;
            }
            float rx = bm_r(u[2]);
            float rt = bm_r(u[3]);
            float ph = 6.2831855f * u2[0];
            int64_t d = pe->n++;
            pe->x[d] = x;
            pe->vx[d] = sgn * (svt * rx);
            pe->vy[d] = svt * (rt * cosf(ph));
            pe->vz[d] = svt * (rt * sinf(ph));
            pe->src_key[n_before[0] + n_inj] = (int)(x * o->inv_r);
            n_inj++;
            pe->m.injected++;
        }
        pe->n_src = n_before[0] + n_inj;
    } else {
        o->sp[0].n_src = n_before[0];
    }
    if (c->n_species > 1) o->sp[1].n_src = n_before[1];
    /* 3. sort   4. deposit   5. field at t_{n+1}   6. MCC */
    for (int s = 0; s < c->n_species; ++s) sort_species(o, s);
    deposit(o);
    field_solve_at(o, o->step + 1u);
    mcc(o);
    coulomb(o);
    o->step += 1u;
}

int oracle_step(orc_t* o, int n_steps) {
    if (!o || n_steps < 0) return -1;
    if (o->loaded_mask != (1 << o->cfg.n_species) - 1) return -1;
    for (int k = 0; k < n_steps; ++k) step_once(o);
    return o->error;
}

/* x in grid-cell units [0, N_c); v in cells/step at t = -dt/2 (R4).  After the
 * last species is loaded: sort, deposit, solve, so that rho/phi/E are valid for step 0. */
int oracle_load_particles(orc_t* o, int s, int64_t n, const float* x, const float* vx,
                          const float* vy, const float* vz) {
    if (!o || s < 0 || s >= o->cfg.n_species || n < 0) return -1;
    if (n > o->cfg.sp[s].capacity) return -2;
    float fNc = (float)o->cfg.n_cells;
    for (int64_t i = 0; i < n; ++i)
        if (!(x[i] >= 0.0f && x[i] < fNc)) return -1;
    orc_species* p = &o->sp[s];
    memcpy(p->x, x, (size_t)n * 4); memcpy(p->vx, vx, (size_t)n * 4);
    memcpy(p->vy, vy, (size_t)n * 4); memcpy(p->vz, vz, (size_t)n * 4);
    p->n = n; p->n_sorted = 0; p->n_src = n;
    memset(&p->m, 0, sizeof(p->m));
    o->loaded_mask |= 1 << s;
    if (o->loaded_mask == (1 << o->cfg.n_species) - 1) {
        o->step = 0; o->error = 0;
        for (int q = 0; q < o->cfg.n_species; ++q) {
            orc_species* pq = &o->sp[q];
            for (int64_t i = 0; i < pq->n; ++i) pq->src_key[i] = (int)(pq->x[i] * o->inv_r);
            sort_species(o, q);
            memset(pq->mask, 0, (size_t)o->cfg.sp[q].capacity);
        }
        deposit(o);
        field_solve_at(o, 0u);
    }
    return 0;
}

int oracle_get_rho_phi_E(orc_t* o, double* rho, double* phi, double* E, int n_nodes) {
    if (!o || n_nodes != o->nodes) return -1;
    if (rho) memcpy(rho, o->rho, (size_t)n_nodes * 8);
    if (phi) memcpy(phi, o->phi, (size_t)n_nodes * 8);
    if (E) memcpy(E, o->E, (size_t)n_nodes * 8);
    return o->error;
}

/* moments over ALL live slots [0, N_s) (sorted part + birth tail); density = rho_s of the
 * last deposit; optional EEDF histogram of E = c_eV |v|^2 on [0, E_max) with n_bins bins. */
int oracle_moments(orc_t* o, int s, orc_moments* out, double* density, int n_density,
                   int64_t* eedf, int n_bins, double E_max) {
    if (!o || s < 0 || s >= o->cfg.n_species || !out) return -1;
    orc_species* p = &o->sp[s];
    orc_moments m = p->m;
    m.count = p->n; m.n_sorted = p->n_sorted;
    m.sum_vx = m.sum_vy = m.sum_vz = m.sum_v2 = m.sum_v4 = 0.0;
    if (eedf) memset(eedf, 0, (size_t)n_bins * 8);
    double c_eV = o->cfg.sp[s].c_eV;
    for (int64_t i = 0; i < p->n; ++i) {
        double vx = p->vx[i], vy = p->vy[i], vz = p->vz[i];
        double g2 = (vx * vx + vy * vy) + vz * vz;
        m.sum_vx += vx; m.sum_vy += vy; m.sum_vz += vz;
        m.sum_v2 += g2; m.sum_v4 += g2 * g2;
        if (eedf) {
            double En = c_eV * g2;
            if (En < E_max) {
                int b = (int)(En / E_max * (double)n_bins);
                if (b >= 0 && b < n_bins) eedf[b]++;
            }
        }
    }
    if (density) {
        if (n_density != o->nodes) return -1;
        memcpy(density, p->rho_s, (size_t)n_density * 8);
    }
    *out = m;
    return o->error;
}

/* ---- debug access for the parity harness ------------------------------------------ */
enum { ORC_X = 0, ORC_VX, ORC_VY, ORC_VZ, ORC_KEYS, ORC_OFFSETS, ORC_MASK, ORC_E32, ORC_RHO_S, ORC_PARTNER };

int64_t oracle_debug_count(orc_t* o, int what, int s) {
    if (!o) return -1;
    switch (what) {
        case ORC_X: case ORC_VX: case ORC_VY: case ORC_VZ: return o->sp[s].n;
        case ORC_KEYS: return o->sp[s].n_src;
        case ORC_OFFSETS: return o->n_sc + 1;
        case ORC_MASK: case ORC_PARTNER: return o->sp[s].n_sorted;
        case ORC_E32: return o->nodes;
        case ORC_RHO_S: return o->nodes;
    }
    return -1;
}

int oracle_debug_get(orc_t* o, int what, int s, void* dst, size_t bytes) {
    if (!o || !dst) return -1;
    int64_t n = oracle_debug_count(o, what, s);
    if (n < 0) return -1;
    const void* src = NULL;
    size_t el = 4;
    orc_species* p = &o->sp[s];
    switch (what) {
        case ORC_X: src = p->x; break;
        case ORC_VX: src = p->vx; break;
        case ORC_VY: src = p->vy; break;
        case ORC_VZ: src = p->vz; break;
        case ORC_KEYS: src = p->src_key; break;
        case ORC_OFFSETS: src = p->offsets; break;
        case ORC_MASK: src = p->mask; el = 1; break;
        case ORC_PARTNER: src = p->partner; break;
        case ORC_E32: src = o->E32; break;
        case ORC_RHO_S: src = p->rho_s; el = 8; break;
    }
    if (bytes < (size_t)n * el) return -1;
    memcpy(dst, src, (size_t)n * el);
    return 0;
}

int oracle_debug_set_E32(orc_t* o, const float* E32, int n_nodes) {
    if (!o || n_nodes != o->nodes) return -1;
    memcpy(o->E32, E32, (size_t)n_nodes * 4);
    return 0;
}

int oracle_n_sort_cells(orc_t* o) { return o ? o->n_sc : -1; }
int oracle_n_nodes(orc_t* o) { return o ? o->nodes : -1; }
uint32_t oracle_step_index(orc_t* o) { return o ? o->step : 0u; }

/* Stand-alone entry for the closed-form pins: runs field_solve() itself -- the function the cycle
 * executes -- on a caller-supplied rho with the wall potentials given directly.  phi and E must
 * hold nodes + 1 doubles (periodic: slot N_c is the wrap node). */
int oracle_solve_field(int n_cells, int bc, const double* rho, double phi0, double phiN,
                       double* phi, double* E) {
    orc_t o;
    memset(&o, 0, sizeof(o));
    o.cfg.n_cells = n_cells; o.cfg.bc = bc;
    o.nodes = bc == 1 ? n_cells : n_cells + 1;
    o.rho = (double*)rho; o.phi = phi; o.E = E;
    o.tmp = calloc((size_t)n_cells + 2, 8);
    o.E32 = calloc((size_t)n_cells + 2, 4);
    field_solve(&o, phi0, phiN);
    free(o.tmp); free(o.E32);
    return 0;
}

/* ====================================================================================================
 * f2 -- the paper's own GAPPED IN-PLACE fine sort (Fig. 2, L63 section 3.2
 * section 3.7, Fig. 6-9), stated step by step: every sort cell owns n_max slots, the first N_i of them
 * valid; the free slots at the end serve as the sorting buffer.
 *   push (fused, L182)  every valid particle is pushed in place
 *   step 1a (L166)      particles that left their cell are copied to the free slots at the END of the
 *                       cell (index counted down from n_max); particles that left the box are dropped
 *   step 1b (L168)      the gaps are closed with the last valid particles of the cell
 *   step 2  (L184)      cell i takes from the rejected buffers of cells i-1 and i+1 what belongs to i
 *   step 3  (L186)      rejected particles that moved farther than one cell go straight to their cell
 * The order inside a cell is undefined in the paper (atomic counters); what IS defined is the result as
 * a multiset: afterwards cell k holds exactly the surviving particles with key k ("all particles are
 * arranged in correct sorting cells", L192).  Pin: that multiset, taken from the compact stable sort of
 * the same particles (sort_species above), tests/test_oracle_gapped.py.  Bounded box only.
 * ==================================================================================================== */
typedef struct {
    int n_cells, n_sc, n_max;
    float inv_r, kappa;
    float *x, *vx, *vy, *vz; /* n_sc * n_max slots each */
    int32_t *N, *R;          /* valid / rejected particles per sort cell */
    float* E32;              /* n_cells + 1 nodes */
    uint8_t* hole;           /* scratch: n_max flags */
    int64_t absorbed_left, absorbed_right, moved_near, moved_far;
    int error;               /* -2: a cell overflowed (particles dropped) */
} orc_gapped;

int oracle_gapped_destroy(orc_gapped* g) {
    if (!g) return 0;
    free(g->x); free(g->vx); free(g->vy); free(g->vz); free(g->N); free(g->R); free(g->E32); free(g->hole);
    free(g);
    return 0;
}

int oracle_gapped_create(int n_cells, double sort_inv_ratio, int n_max, double kappa, orc_gapped** out) {
    if (!out || n_cells < 2 || n_max < 1 || !(sort_inv_ratio > 0.0)) return -1;
    orc_gapped* g = (orc_gapped*)calloc(1, sizeof(orc_gapped));
    g->n_cells = n_cells; g->n_max = n_max; g->kappa = (float)kappa; g->inv_r = (float)sort_inv_ratio;
    g->n_sc = (int)ceil((double)n_cells * sort_inv_ratio);
    size_t tot = (size_t)g->n_sc * (size_t)n_max;
    g->x = malloc(tot * 4); g->vx = malloc(tot * 4); g->vy = malloc(tot * 4); g->vz = malloc(tot * 4);
    g->N = calloc((size_t)g->n_sc, 4); g->R = calloc((size_t)g->n_sc, 4);
    g->E32 = calloc((size_t)n_cells + 2, 4);
    g->hole = malloc((size_t)n_max);
    *out = g;
    return 0;
}

static int gapped_key(const orc_gapped* g, float x) { /* -1 / -2: left the box (L41) */
    if (!(x >= 0.0f && x < (float)g->n_cells)) return x < 0.0f ? -1 : -2;
    return (int)(x * g->inv_r);
}

static void gapped_put(orc_gapped* g, size_t dst, size_t src) {
    g->x[dst] = g->x[src]; g->vx[dst] = g->vx[src]; g->vy[dst] = g->vy[src]; g->vz[dst] = g->vz[src];
}

/* append to cell k behind its valid particles, in front of its rejected buffer */
static void gapped_append(orc_gapped* g, int k, size_t src) {
    if (g->N[k] >= g->n_max - g->R[k]) { g->error = -2; return; }
    gapped_put(g, (size_t)k * g->n_max + (size_t)g->N[k], src);
    g->N[k]++;
}

int oracle_gapped_load(orc_gapped* g, int64_t n, const float* x, const float* vx, const float* vy, const float* vz) {
    if (!g) return -1;
    memset(g->N, 0, (size_t)g->n_sc * 4); memset(g->R, 0, (size_t)g->n_sc * 4);
    g->absorbed_left = g->absorbed_right = g->moved_near = g->moved_far = 0; g->error = 0;
    for (int64_t i = 0; i < n; ++i) {
        int k = gapped_key(g, x[i]);
        if (k < 0) return -1;
        if (g->N[k] >= g->n_max) { g->error = -2; continue; }
        size_t d = (size_t)k * g->n_max + (size_t)g->N[k]++;
        g->x[d] = x[i]; g->vx[d] = vx[i]; g->vy[d] = vy[i]; g->vz[d] = vz[i];
    }
    return g->error;
}

int oracle_gapped_set_E32(orc_gapped* g, const float* E32, int n_nodes) {
    if (!g || n_nodes != g->n_cells + 1) return -1;
    memcpy(g->E32, E32, (size_t)n_nodes * 4);
    return 0;
}

int oracle_gapped_step(orc_gapped* g) {
    if (!g) return -1;
    int nm = g->n_max;
    /* push + step 1a + step 1b, cell by cell */
    for (int c = 0; c < g->n_sc; ++c) {
        size_t base = (size_t)c * nm;
        int N = g->N[c], top = nm, holes = 0;
        for (int j = 0; j < N; ++j) {
            gather_push(g->E32, g->kappa, g->n_cells, 0, &g->x[base + j], &g->vx[base + j]);
            int k = gapped_key(g, g->x[base + j]);
            g->hole[j] = 0;
            if (k == c) continue;
            g->hole[j] = 1; ++holes;
            if (k == -1) { g->absorbed_left++; continue; }
            if (k == -2) { g->absorbed_right++; continue; }
            if (top - 1 < N) { g->error = -2; continue; }       /* no free slot left at the end of the cell */
            --top;                                               /* step 1a: N_index counts down (L166) */
            gapped_put(g, base + top, base + j);
        }
        int V = N - holes, last = N - 1;                          /* step 1b: close the gaps from the end */
        for (int j = 0; j < V; ++j) {
            if (!g->hole[j]) continue;
            while (g->hole[last]) --last;
            gapped_put(g, base + j, base + last);
            --last;
        }
        g->N[c] = V; g->R[c] = nm - top;
    }
    /* step 2: what the neighbours rejected and belongs here (L184) */
    for (int c = 0; c < g->n_sc; ++c)
        for (int d = -1; d <= 1; d += 2) {
            int nb = c + d;
            if (nb < 0 || nb >= g->n_sc) continue;
            size_t nbase = (size_t)nb * nm;
            for (int q = nm - g->R[nb]; q < nm; ++q)
                if (gapped_key(g, g->x[nbase + q]) == c) { gapped_append(g, c, nbase + q); g->moved_near++; }
        }
    /* step 3: the rare particles that moved farther than one cell (L186) */
    for (int c = 0; c < g->n_sc; ++c) {
        size_t base = (size_t)c * nm;
        for (int q = nm - g->R[c]; q < nm; ++q) {
            int k = gapped_key(g, g->x[base + q]);
            if (k == c - 1 || k == c + 1) continue;
            gapped_append(g, k, base + q); g->moved_far++;
        }
    }
    for (int c = 0; c < g->n_sc; ++c) g->R[c] = 0;               /* the buffers are free again */
    return g->error;
}

/* copies the gapped arrays (n_sc * n_max slots) and the counts; stats = {absorbed_left, absorbed_right,
 * moved_near, moved_far} */
int oracle_gapped_get(orc_gapped* g, int32_t* N, float* x, float* vx, float* vy, float* vz, int64_t* stats) {
    if (!g) return -1;
    size_t tot = (size_t)g->n_sc * (size_t)g->n_max;
    if (N) memcpy(N, g->N, (size_t)g->n_sc * 4);
    if (x) memcpy(x, g->x, tot * 4);
    if (vx) memcpy(vx, g->vx, tot * 4);
    if (vy) memcpy(vy, g->vy, tot * 4);
    if (vz) memcpy(vz, g->vz, tot * 4);
    if (stats) { stats[0] = g->absorbed_left; stats[1] = g->absorbed_right; stats[2] = g->moved_near; stats[3] = g->moved_far; }
    return g->error;
}
int oracle_gapped_n_sort_cells(orc_gapped* g) { return g ? g->n_sc : -1; }
