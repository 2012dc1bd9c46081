/*
 * pic1d_gsort.h -- C-ABI of the paper's own GAPPED IN-PLACE fine sort fused with the pusher (
 * PAPER.md L55 Fig. 2, L63 section 3.2, L160-192 section 3.7, Fig. 6-9), as a second push + sort back-end next
 * to the compact histogram / scan / scatter of pic1d.h.  It is the design for species that obey Eq. 5 (L162:
 * "only a small number of particles leaves its sorting cell during one time step"): every particle is pushed
 * in place (16 B per particle-step) and only the movers are copied, instead of the 8 + 32 B per particle-step
 * of the compact two-pass sort.
 *
 * Layout: every sort cell owns n_max slots of four fp32 SoA arrays (x, vx, vy, vz; cell k = slots k n_max ..
 * (k+1) n_max - 1); the first N_i[k] are valid, the free slots at the end are the sorting buffer.  One step =
 *   kernel 1: gather + leapfrog push (L150-156) + step 1a (rejected particles to the end of the cell, L166)
 *             + step 1b (gaps closed with the last valid particles, L168); particles that left the box are removed
 *   kernel 2: step 2 -- cell i collects from the rejected buffers of cells i-1 and i+1 (L184)
 *   kernel 3: step 3 -- the rare particles that moved farther than one cell (L186)
 * The order of the particles inside a cell is NOT defined (the paper assigns slots with atomic counters); what is
 * defined, and what the tests compare with the oracle, is the multiset of particles of every cell and N_i.
 * Bounded box with absorbing walls; the field is the caller's (fp32, n_cells + 1 nodes, normalised units of
 * pic1d.h).  All device memory is one caller-owned workspace; kernels run on the caller's stream.
 * Returns 0 or a negative PIC1D_ERR_* code of pic1d.h.
 */
#ifndef PIC1D_GSORT_H_
#define PIC1D_GSORT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pic1d_gsort pic1d_gsort_t; /* opaque */

/* bytes of device workspace for n_cells grid cells, sort cells of 1 / sort_inv_ratio grid cells (a power of two,
 * as in pic1d_config_t) and n_max <= 8192 slots per sort cell.  HOST pointer. */
int pic1d_gsort_workspace_bytes(int n_cells, double sort_inv_ratio, int n_max, size_t* bytes_out);

/* workspace: DEVICE, 256-byte aligned, caller-owned; kappa: the species' signed push constant (Eq. 3) */
int pic1d_gsort_create(int n_cells, double sort_inv_ratio, int n_max, double kappa, void* workspace,
                       size_t workspace_bytes, void* cuda_stream, pic1d_gsort_t** out);

/* distribute n particles (x in [0, n_cells)) over the sort cells; HOST (on_device = 0, synchronises) or DEVICE
 * arrays, copied.  A cell that would need more than n_max slots -> sticky PIC1D_ERR_CAPACITY. */
int pic1d_gsort_load(pic1d_gsort_t* h, int64_t n, const float* x, const float* vx, const float* vy,
                     const float* vz, int on_device);

/* the fp32 field the push gathers: n_nodes = n_cells + 1 values, HOST or DEVICE, copied */
int pic1d_gsort_set_E32(pic1d_gsort_t* h, const float* E32, int n_nodes, int on_device);

/* enqueue n_steps of push + gapped sort (three kernels each); asynchronous */
int pic1d_gsort_step(pic1d_gsort_t* h, int n_steps);

/* copy to HOST (synchronises; any pointer may be NULL): N_i[n_sort_cells]; the four gapped arrays
 * (n_sort_cells * n_max floats each); stats[5] = particles absorbed at the left / right wall, moved by step 2,
 * moved by step 3 (cumulative since the load), sticky error (0 or PIC1D_ERR_CAPACITY: a cell overflowed and
 * particles were dropped).  Returns the sticky error. */
int pic1d_gsort_get(pic1d_gsort_t* h, int32_t* N_i, float* x, float* vx, float* vy, float* vz, int64_t* stats);

int pic1d_gsort_n_sort_cells(const pic1d_gsort_t* h);
int pic1d_gsort_destroy(pic1d_gsort_t* h);

#ifdef __cplusplus
}
#endif
#endif /* PIC1D_GSORT_H_ */
