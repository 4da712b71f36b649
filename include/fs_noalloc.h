/* fs_noalloc.h -- ONE entry point of libfs.so that allocates nothing: the continuity check of the projected field.
 *
 * For callers that cannot call cudaMalloc or hand over a workspace (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid allocation).  Every other call of the library works on a grid whose device memory is the workspace
 * the caller passed to fs_grid_create (include/fs.h); this one needs no grid and no workspace: its reduction scratch is a
 * file-scope static __device__ array inside the library (128.25 KB; every GPU that loads libfs.so holds it until exit).
 *
 * What it computes: the discrete divergence of a staggered velocity field on a uniform, triply periodic box, the quantity
 * the projection step drives to zero (Eq. 2 / Eq. 6), and its maximum norm and
 * squared 2-norm -- the same numbers fs_step_info.max_abs_div and fs_fields_get(FS_DIV) give on a grid:
 *
 *   div(i,j,k) = (u(i+1,j,k) - u(i,j,k)) / hx + (v(i,j+1,k) - v(i,j,k)) / hy + (w(i,j,k+1) - w(i,j,k)) / hz   (indices wrap)
 *   result[0]  = max |div|,   result[1] = sum div^2   (both accumulated in fp64, added in a fixed order: deterministic)
 *
 * Layout: u, v, w, div are nx*ny*nz words each, x fastest, then y, then z; u(i,j,k) is the velocity on the face at
 * x0 + i hx of cell (i,j,k) (the library's layout of a periodic direction, fs.h "Layout").
 *
 * Limit: nx * ny * nz <= FS_NOALLOC_MAX_CELLS (the scratch holds one pair of partials per 2048 cells).  A larger box is
 * rejected with FS_ERR_UNSUPPORTED and a line on stderr; nothing is launched.
 *
 * Sharing: every call on a device uses the same scratch array, which keeps the last call's contents.  The call clears the
 * word that must start at zero (the arrival counter) on the caller's stream before the kernel; partials are overwritten
 * before they are read.  Calls that OVERLAP on the GPU (two streams, two host threads, two graphs in flight) race on the
 * scratch and give undefined results: serialise them on one stream or with events.
 *
 * The first call on each device looks up the scratch array's device address (cudaGetSymbolAddress, with that device
 * current) and caches it; the call never calls cudaMalloc, cudaFree or an allocating library routine.
 */
#ifndef FS_NOALLOC_H
#define FS_NOALLOC_H
#include "fs.h"

#ifdef __cplusplus
extern "C" {
#endif

#define FS_NOALLOC_MAX_CELLS 16777216LL /* 256^3; c1-c4 of BASELINE.json fit, c5 (512^3) does not */

/* u, v, w:   DEVICE pointers (on the CURRENT device), nx*ny*nz words of `dtype`, read only.
 * div_out:   DEVICE pointer, nx*ny*nz words of `dtype`, written; NULL = do not store the field.
 * result:    DEVICE pointer, 2 doubles, written: { max |div|, sum div^2 }.
 * stream:    cudaStream_t the work is enqueued on (NULL = the legacy default stream).  Asynchronous: returns after the
 *            launch; outputs are valid once the stream reaches this point.
 * Returns FS_OK; FS_ERR_INVALID_ARG (NULL input / result, a size < 1, a spacing <= 0, a pointer that is not device memory
 * of the current device), FS_ERR_UNSUPPORTED (more than FS_NOALLOC_MAX_CELLS cells), FS_ERR_CUDA (the symbol lookup or the
 * launch failed).  Outputs are untouched on failure.  Caller owns all five buffers. */
fs_status fs_divergence_noalloc(int nx, int ny, int nz, double hx, double hy, double hz, fs_dtype dtype,
                                const void* u, const void* v, const void* w, void* div_out, double* result,
                                void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
