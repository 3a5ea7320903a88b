/*
 * sg_disk_static.h -- one entry point of the sg_disk library that never allocates device memory.
 *
 * Who this is for.  Everything in sg_disk.h works through a context that sg_create fills with cudaMalloc'ed arrays
 * (vertex lists, tiles, tables, partial sums).  Some host codes cannot do that:
 *   - a hydrodynamics code whose own arena already holds the whole device: a cudaMalloc from a library may simply
 *     fail there, and the code has no way to lend the library a piece of its arena through sg_create;
 *   - a caller inside a time-step loop that must not stall: cudaMalloc and cudaFree synchronise the device and take
 *     a driver lock, so a library that allocates behind the caller's back serialises every stream the caller runs;
 *   - a plug-in or analysis hook that the host application calls with the rule "no allocation in here"
 *     (fixed memory budget accounted up front, or an allocator the library is not allowed to bypass).
 * For them sg_force_uniform_static computes the zeroth-order force sum of the paper on ONE uniform grid with nothing
 * but the caller's three arrays and a fixed work array that lives inside the library image.
 *
 * What it computes (PAPER.md:57-69 Eq. 4-5, :86-94; same sum as sg_set_density + sg_force on a one-level layout):
 *     Fx_t = G * sum_c sigma_c * [[ -ln( (ybar-y_t) + r ) ]]_c ,   Fy_t the same with x and y exchanged,
 * at the centre of every cell t of an nx x ny grid of square cells, the sum running over all cells c (t included).
 * It is the vertex-regrouped direct sum of the library's interaction kernel (one sqrt and two ln per
 * (target, vertex) pair), written for a uniform grid: the signed vertex weights w_v -- the scratch data of that
 * kernel -- go to the library's static array instead of a cudaMalloc'ed one.  On a uniform grid no cell centre lies
 * on a grid line, so the modified primitive of PAPER.md:96-100 never applies.  The result does not depend on the cell
 * width (the integrals are dimensionless), hence no width argument.
 *
 * The static work array
 *   - SG_STATIC_MAX_VERTICES doubles (528,392 bytes), a file-scope __device__ array of libsg_disk.so.  Every GPU on
 *     which the process loads the library's device code holds these bytes until the process exits, whether this entry
 *     point is used or not.  That is why the limit is modest.
 *   - Limit: (nx + 1) * (ny + 1) <= SG_STATIC_MAX_VERTICES, i.e. up to 256 x 256 cells (or e.g. 512 x 127), and
 *     nx, ny <= SG_STATIC_MAX_SIDE.  Larger grids are refused with SG_ERR_ARG and a message; use the context API
 *     for them.
 *   - The first call on a device looks up the array's device address (cudaGetSymbolAddress, with that device current)
 *     and keeps it; this is host-side set-up that talks to the driver, so make the first call on each device early,
 *     outside any stream capture.  Later calls only enqueue two kernels.
 *   - ALL calls on one device share the one array and it keeps whatever the previous call left.  Nothing in it has to
 *     start at zero: each call first overwrites the (nx+1)*(ny+1) weights it is going to read and reads no others, so
 *     neither stale weights of an earlier, larger grid nor a freshly loaded (zero) array change the result.
 *     Two calls whose kernels can overlap on the GPU (different streams without an ordering event between them,
 *     or two host threads each with its own stream) race on the array and give wrong forces: order them yourself.
 *     Calls enqueued on one stream are ordered by the stream and are safe.
 *
 * The call itself performs no cudaMalloc, cudaFree, cudaMallocAsync or other allocating CUDA / library routine, and
 * no device synchronisation: argument checks, the one-time address look-up, two kernel launches on cuda_stream.
 */
#ifndef SG_DISK_STATIC_H
#define SG_DISK_STATIC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SG_STATIC_MAX_VERTICES 66049   /* 257 * 257: up to 256 x 256 cells */
#define SG_STATIC_MAX_SIDE 1024        /* longest side of an elongated grid (size of an in-kernel ln table) */

/*
 *   nx, ny        cells along x and y, each in [1, SG_STATIC_MAX_SIDE], (nx+1)*(ny+1) <= SG_STATIC_MAX_VERTICES
 *   G             gravitational constant multiplying the sums (finite)
 *   sigma_dev     device [ny][nx] FP64, x fastest: surface density of cell (i, j); read only
 *   Fx_dev, Fy_dev  device [ny][nx] FP64, same order; written.  Must not alias sigma_dev.
 *   device        CUDA device ordinal the three arrays live on (the caller's current device is left unchanged)
 *   cuda_stream   a cudaStream_t passed as void*, NULL = default stream; the work is asynchronous on it and the
 *                 arrays must stay alive until it has drained
 * Returns SG_OK, SG_ERR_ARG (null pointer, bad or too large size, G not finite) or SG_ERR_CUDA (0 / -1 / -3 of
 * sg_disk.h); sg_static_last_error() has the message of the calling thread's last failure.
 * Deterministic: same inputs, same bits (fixed summation order, no atomics).
 */
int sg_force_uniform_static(int nx, int ny, double G, const double *sigma_dev, double *Fx_dev, double *Fy_dev,
                            int device, void *cuda_stream);

const char *sg_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SG_DISK_STATIC_H */
