/* nh_noalloc.h -- two lattice-Boltzmann steps for callers that must not allocate memory.
 *
 * Who this is for.  The normal path (include/nh.h) builds a lattice handle: nh_init_lattice takes a device workspace from
 * the caller, but it also creates host objects, a pinned host word (cudaHostAlloc) and, on demand, CUDA events and graphs.
 * Some hosts cannot afford any of that at the point where they want LB steps done:
 *   - a solver plugged into an application that reserved the whole device for its own memory pool at start-up, so a
 *     later cudaMalloc from a library either fails or steals from that pool;
 *   - a time-critical loop (in-situ coupling to an instrument or to another solver), where cudaMalloc / cudaFree are
 *     off limits because they take the driver's global lock and wait for the device to go idle;
 *   - code that runs under an allocation audit ("nothing allocates after initialisation").
 * For them the one call below advances a population array by TWO LB steps and allocates nothing: no cudaMalloc,
 * cudaFree, cudaHostAlloc, no event, graph or stream creation, no library call that allocates, and no host heap on the
 * success path.  Inputs and outputs are the caller's device arrays.
 *
 * Where the scratch lives.  The two-step kernel (csrc/nh_lb2.cuh: Eqs. 14-23, two steps per pass over
 * HBM) needs memory that is neither input nor output: a ring of z-planes of post-collision populations between its
 * two phases, per-piece progress flags, a ticket counter and the unit order table.  Here they sit in ONE array of
 * NH_NOALLOC_SCRATCH_BYTES bytes that is part of the library image itself (a file-scope `static __device__` array in
 * csrc/nh_noalloc.cu).  The price: every GPU on which this library's code gets loaded holds these 16 MiB until the
 * process exits, whether or not the call is ever used.
 *
 * The limit.  A lattice fits when the control block and at least three ring planes fit:
 *     256-rounded 8 * (40 + 2 (nz-2) c + (nz-2))  +  R * 19 * nx * (ny+2) * word  <=  NH_NOALLOC_SCRATCH_BYTES,
 *     c = pieces per ring plane = ceil((ny+2) nx / 256) for nx <= 256, (ny+2) nx / 256 otherwise,  word = 4 or 8 bytes,
 * with R = min(8, nz-2) shrunk down to 3 if need be.  In round numbers: planes of up to about 70 000 cells in FP32
 * (256x256 fits, with R = 3) and 35 000 in FP64 (128x256).  Larger lattices are refused with NH_EINVAL and a message
 * that states the bytes needed; they belong on the handle path, whose workspace the caller sizes.
 */
#ifndef NH_NOALLOC_H
#define NH_NOALLOC_H
#include <stddef.h>
#include "nh.h"
#ifdef __cplusplus
extern "C" {
#endif

#define NH_NOALLOC_SCRATCH_BYTES (16u * 1024u * 1024u)

/* f_out := two LB steps applied to f_in (collide with Guo forcing, stream, half-way bounce-back at the plates z = 0 and
 * z = nz-1, periodic x and y; the same arithmetic, bit for bit, as two LB steps of nh_step with the force frozen).
 *
 *   nx, ny, nz   grid, nz counting the two plate layers.  nx must be 64, 128 or a multiple of 256 (the kernel's pieces are
 *                256 consecutive cells); nz >= 5; 19*nx*ny*nz < 2^31; and the lattice must fit the scratch (above).
 *   precision    NH_FP64_SHIFTED .. NH_FP64_UNSHIFTED: storage type and form of the populations (include/nh.h).
 *   tau          SRT relaxation time, > 0.5.   g[3]: body acceleration, HOST pointer.
 *   f_in_dev     DEVICE, [19][nz][ny][nx] words of the precision's type: the post-collision populations the next step
 *                gathers from -- the layout of NH_FIELD_POPULATIONS (what nh_get_rows of all ny rows packs).  Read only.
 *   F_lc_dev     DEVICE, [3][nz][ny][nx], the force density F^LC held fixed over both steps, or NULL
 *                for none.  Read only.
 *   f_out_dev    DEVICE, same shape as f_in_dev, must not overlap it.  Only the fluid layers z = 1 .. nz-2 are written;
 *                the two plate layers keep whatever they held.
 *   cuda_stream  cudaStream_t the work is queued on (NULL: the legacy default stream).  It must belong to the device
 *                that is current in the calling thread, and the three arrays must live on that device.
 *
 * The call returns after the work has finished (it synchronises the stream), so its return code covers the kernels:
 * NH_OK; NH_EINVAL for a bad argument or a lattice beyond the limit (nothing has been launched); NH_ECUDA if a CUDA call
 * failed, there is no device, or a dependency wait inside the kernel ran into its 4 s bound (f_out is then garbage).
 * The text is in nh_last_error().
 *
 * First call on each device.  The array's device address is looked up once per device (cudaGetSymbolAddress, with that
 * device current) and remembered; loading the kernels is also paid there.  Make that first call early, during your own
 * set-up, and before any stream capture is begun.
 *
 * Sharing.  There is one scratch array per device, and every call uses all of it and finds the previous call's
 * contents in it.  The call clears the part that must start from zero (ticket, flags, counters, error word) itself, on
 * the stream, before the main kernel.  Two calls whose work overlaps in time on one GPU -- different streams, different
 * host threads, different processes' contexts do NOT count, each context has its own copy -- would race on the ring and
 * the flags: issue them one after the other.  Lattices made by nh_init_lattice never touch this array. */
int nh_lb_two_steps_noalloc(int nx, int ny, int nz, int precision, double tau, const double* g,
                            const void* f_in_dev, const void* F_lc_dev, void* f_out_dev, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
