/*
 * pic1d_static.h -- the Poisson + E solve of the PIC cycle (Eq. 1-2; Thomas elimination,
 * L142-146) as a stand-alone call that creates no device memory at all.
 *
 * Who this is for.  Everything else in this library works out of a workspace the caller allocates
 * (pic1d_workspace_bytes / pic1d_create).  Some callers cannot do that: a host code whose own memory manager has
 * already claimed the whole GPU (a cudaMalloc from anybody else then simply fails), a plug-in that is handed
 * nothing but the input and output buffers of its host application and has no allocator of its own, or a
 * time-step loop that must never run into the device-wide synchronisation a cudaMalloc / cudaFree implies.
 * Such a caller owns rho, phi and E anyway -- but the solver also needs two temporary arrays of n_cells doubles
 * (the running sums S and T below), and there is nobody to provide them.  Here they live in a fixed array that is
 * part of the library image itself (a file-scope `static __device__` array in csrc/pic1d_field_static.cu), so the
 * call allocates nothing: no cudaMalloc, no cudaFree, no library routine that allocates.
 *
 * The price, and the limit.  The array has a fixed size: grids of up to PIC1D_FIELD_STATIC_MAX_CELLS = 65536
 * cells, i.e. 2 x 65536 x 8 B = 1 MiB of device memory, which EVERY GPU that loads libpic1d.so's device code
 * holds from that moment until the process exits, whether this call is ever made there or not (when exactly the
 * CUDA runtime loads the code -- with the library or at the first use -- is its module-loading policy, not ours).
 * Larger grids are refused (PIC1D_ERR_ARG); use pic1d_create with a workspace for those.
 *
 * What it computes (identical arithmetic to the field kernel of pic1d_step for grids above 24576 cells):
 *   phi[j-1] - 2 phi[j] + phi[j+1] = -rho[j]  (Eq. 1 in the normalised units of pic1d.h, L113-117),
 *   E[j] = (phi[j-1] - phi[j+1]) / 2          (Eq. 2), with the half-cell Gauss law at the two wall nodes,
 * solved as the Thomas recurrences of L142 summed in closed form: S_m = sum_{i=1..m} rho_i, T_m = sum_{i=1..m} S_i,
 * d_1 = (phi_N - phi_0 + T_{N-1}) / N, phi_j = phi_0 + j d_1 - T_{j-1}, E_j = -d_1 + (S_{j-1} + S_j) / 2.
 * One thread block, two fp64 prefix sums, no host round trip (contrast L144).
 */
#ifndef PIC1D_STATIC_H_
#define PIC1D_STATIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIC1D_FIELD_STATIC_MAX_CELLS 65536

/*
 * Solve for phi and E on the current CUDA device, enqueued on cuda_stream (a cudaStream_t of the CURRENT device;
 * NULL = default stream).  Asynchronous: returns once the kernel is enqueued.
 *
 *   rho      DEVICE, fp64, n_nodes values, read only: net charge density, raw linear-weighting sums exactly as
 *            pic1d_get_rho_phi_E returns them (no wall-node doubling).  n_nodes = n_cells + 1 for bc = 0
 *            (bounded, walls at nodes 0 and n_cells), n_cells for bc = 1 (periodic; the mean of rho is removed
 *            before solving and phi is returned with zero mean).
 *   phi, E   DEVICE, fp64, n_nodes values each, written.  Must not overlap rho or each other.
 *   E32      DEVICE, fp32, n_nodes values, written (the copy of E a pusher gathers), or NULL.
 *   n_cells  2 .. PIC1D_FIELD_STATIC_MAX_CELLS.
 *   bc       0 bounded, 1 periodic.
 *   phi0     potential of the left wall, phi[0] (bc = 0; the right wall is phi[n_cells] = 0, as everywhere in
 *            pic1d.h).  Ignored for bc = 1.
 * The caller keeps ownership of every buffer and keeps them alive until the stream has run the kernel.
 *
 * Returns 0, PIC1D_ERR_ARG (-1: a NULL rho / phi / E, bc not 0 or 1, phi0 not finite, n_cells below 2 or above
 * the maximum -- nothing has been enqueued) or PIC1D_ERR_CUDA (-3: looking up the scratch array or the launch
 * failed).  pic1d_field_solve_static_error() then says which, in words.
 *
 * Set-up on first use.  The first call a host process makes on a given device asks the CUDA runtime where that
 * device keeps its copy of the scratch array (cudaGetSymbolAddress, with that device current) and remembers the
 * answer; this may make the runtime load the library's device code onto the GPU.  Make that first call early,
 * during start-up and before any stream capture begins; later calls on the same device only launch the kernel.
 *
 * Sharing.  There is ONE scratch array per device, shared by every call, every stream and every host thread of
 * the process.  It keeps whatever the previous call left in it; that is harmless, because a call writes every
 * element of S and T before it reads it -- nothing has to start at zero, so nothing is cleared.  But two calls
 * whose kernels can run at the same time on one GPU (different streams without an event between them, or two
 * host threads) overwrite each other's sums and both results are garbage: put all calls of a device on one
 * stream, or order them with events.  Calls on different GPUs never interfere.
 */
int pic1d_field_solve_static(const double* rho, double* phi, double* E, float* E32, int n_cells, int bc,
                             double phi0, void* cuda_stream);

/* Text of the last failure of pic1d_field_solve_static on the calling host thread ("" if none so far).  The
 * pointer stays valid until that thread's next failing call.  HOST. */
const char* pic1d_field_solve_static_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PIC1D_STATIC_H_ */
