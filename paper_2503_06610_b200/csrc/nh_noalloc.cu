// nh_noalloc.cu -- nh_lb_two_steps_noalloc (include/nh_noalloc.h): the two-step LB kernel of nh_lb2.cuh for callers that
// may not allocate.  Everything the kernel needs besides its inputs and outputs -- plane ring, progress flags, ticket,
// order table, error word -- lives in the file-scope device array below instead of in a caller-sized workspace.
//
// The arithmetic is nh_lb2.cuh's, untouched (Eqs. 14-23; bounce-back PAPER.md:141; periodic x, y
// PAPER.md:225); this file only lays the scratch out, clears what has to start from zero and launches.
//
// Rules this file keeps:
//   - no cudaMalloc / cudaFree / cudaHostAlloc / event / graph / stream creation, no allocating library call; on the
//     success path no host heap either (error texts go through std::string in nh_api.cu);
//   - in HOST code `g_scratch` is only a handle for the runtime, not an address a kernel could use: the device address
//     comes from cudaGetSymbolAddress, asked once per device with that device current, and that is what gets passed;
//   - one array per device, shared by all calls, holding the last call's leftovers: the prepare kernel zeroes the
//     control block on the stream before the main kernel; calls that overlap on the GPU would race (documented).
#include "../../include/nh_noalloc.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <mutex>

#include "nh_internal.h"
#include "nh_lb2.cuh"

namespace {

// The scratch: part of the library image, so every GPU that loads this code holds it until the process ends.
static __device__ __align__(256) unsigned char g_scratch[NH_NOALLOC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_lock;
void* g_scratch_addr[MAX_DEVICES];      // device address of g_scratch on device d, nullptr: not asked yet

constexpr int NT = 128, U = 2;          // CTA shape of the kernel: pieces of NT * U = 256 consecutive cells
constexpr size_t HEADER_WORDS = 8;      // word 0: ticket, word 1: error word; the rest unused
constexpr size_t ALIGN = 256;

int cuda_fail(cudaError_t e, const char* what) {
  char msg[256];
  std::snprintf(msg, sizeof msg, "nh_lb_two_steps_noalloc: %s: %s", what, cudaGetErrorString(e));
  return nh::set_error(NH_ECUDA, msg);
}
int bad(const char* why) {
  char msg[320];
  std::snprintf(msg, sizeof msg, "nh_lb_two_steps_noalloc: %s", why);
  return nh::set_error(NH_EINVAL, msg);
}

// Device address of the scratch on the CURRENT device; the first call per device asks the runtime for it.
int scratch_of_current_device(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e, "cudaGetDevice (no CUDA device? this library has no CPU path)"); }
  if (dev < 0 || dev >= MAX_DEVICES) return bad("device ordinal beyond 63");
  std::lock_guard<std::mutex> hold(g_setup_lock);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_scratch);
    if (e != cudaSuccess || !p) { cudaGetLastError(); return cuda_fail(e, "cudaGetSymbolAddress(scratch)"); }
    g_scratch_addr[dev] = p;
  }
  *out = (unsigned char*)g_scratch_addr[dev];
  return NH_OK;
}

// How one lattice uses the scratch.
struct Plan {
  unsigned cps, ppr, rows_per_piece, pieces2;
  int spr_shift, nzf, D, R;
  unsigned order_len;
  size_t flag_words;      // per phase
  size_t ctrl_bytes;      // header + strip counters + flags + order table, rounded to 256
  size_t plane_bytes;     // one ring plane: 19 * nx * (ny + 2) words
};

// Clears the control block (everything up to the order table) and writes the order table: round j emits phase 2 of
// plane j-D-1, then phase 1 of plane j, so that every unit comes after everything it waits for (nh_lb2.cuh).
__global__ void noalloc_prepare_kernel(unsigned long long* ctrl, unsigned zero_words, unsigned* order, int nzf, int D) {
  const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  for (unsigned w = i; w < zero_words; w += gridDim.x * blockDim.x) ctrl[w] = 0ull;
  if (i == 0) {
    unsigned at = 0;
    for (int j = 0; j < nzf + D + 1; ++j) {
      const int k2 = j - D - 1;
      if (k2 >= 0 && k2 < nzf) order[at++] = 0x80000000u | (unsigned)k2;
      if (j < nzf) order[at++] = (unsigned)j;
    }
  }
}

template <typename T, bool SH>
int run(int nx, int ny, int nz, double tau, const double* g, const void* f_in, const void* F, void* f_out,
        cudaStream_t stream, unsigned char* scratch, const Plan& P) {
  nh::Geom G;
  G.nx = nx; G.ny = ny; G.nz = nz;
  G.plane = (unsigned)nx * ny;
  G.nfluid = G.plane * (unsigned)(nz - 2);
  G.N = (size_t)G.plane * nz;
  nh::LbConst<T> C;
  C.omega = (T)(1.0 / tau);
  C.somega = (T)(1.0 - 1.0 / (2.0 * tau));
  C.gx = (T)g[0]; C.gy = (T)g[1]; C.gz = (T)g[2];
  C.use_flc = F ? 1 : 0;

  unsigned long long* ctrl = (unsigned long long*)scratch;
  nh::Wave W;
  W.ticket = ctrl;                                   // cleared by the prepare kernel: this launch's tickets start at 0
  W.ticket_base = 0;
  W.err = (volatile int*)(ctrl + 1);                 // device memory here (the handle path uses a host-mapped word)
  W.timeout_cycles = 8000000000ll;                   // about 4 s of SM clocks per wait
  W.fault = 0ull;
  W.strip_done = ctrl + HEADER_WORDS;
  W.flag1 = W.strip_done + nh::WAVE_MAX_STRIPS;
  W.flag2 = W.flag1 + P.flag_words;
  unsigned* order = (unsigned*)(W.flag2 + P.flag_words);
  W.order = order;
  W.epoch0 = 1;                                      // one strip: its flags carry 1, cleared flags 0
  W.strip_target[0] = (unsigned long long)P.nzf * P.pieces2;
  for (int s = 1; s < nh::WAVE_MAX_STRIPS; ++s) W.strip_target[s] = 0;
  W.nzf = P.nzf; W.YS = (unsigned)ny; W.nstrips = 1;
  W.cps = P.cps; W.ppr = P.ppr; W.rows_per_piece = P.rows_per_piece;
  W.units_per_strip = P.order_len * P.cps;
  W.rplane = (unsigned)(ny + 2) * (unsigned)nx;
  W.spr_shift = P.spr_shift;
  W.D = P.D; W.R = P.R;
  W.reverse = 0;

  nh::DirTab<const T> A;
  nh::DirTab<T> Rg, B;
  T* ring = (T*)(scratch + P.ctrl_bytes);
  for (int i = 0; i < nh::Q; ++i) {
    A.p[i] = (const T*)f_in + (size_t)i * G.N;
    B.p[i] = (T*)f_out + (size_t)i * G.N;
    Rg.p[i] = ring + (size_t)i * P.R * W.rplane;
  }

  const unsigned zero_words = (unsigned)(HEADER_WORDS + nh::WAVE_MAX_STRIPS + 2 * P.flag_words);
  noalloc_prepare_kernel<<<(zero_words + 255) / 256, 256, 0, stream>>>(ctrl, zero_words, order, P.nzf, P.D);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, "launch of the prepare kernel");
  nh::lb_wave_kernel<T, SH, U, NT><<<W.units_per_strip, NT, 0, stream>>>(A, Rg, B, (const T*)F, G, C, W);
  e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, "launch of the two-step kernel");
  int stalled = 0;
  e = cudaMemcpyAsync(&stalled, ctrl + 1, sizeof(int), cudaMemcpyDeviceToHost, stream);
  if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync(error word)");
  e = cudaStreamSynchronize(stream);
  if (e != cudaSuccess) return cuda_fail(e, "cudaStreamSynchronize");
  if (stalled)
    return nh::set_error(NH_ECUDA, "nh_lb_two_steps_noalloc: a wavefront dependency wait timed out; f_out is invalid "
                                   "(were two calls running on this GPU at once?)");
  return NH_OK;
}

}  // namespace

extern "C" int nh_lb_two_steps_noalloc(int nx, int ny, int nz, int precision, double tau, const double* g,
                                       const void* f_in_dev, const void* F_lc_dev, void* f_out_dev, void* cuda_stream) {
  if (!g || !f_in_dev || !f_out_dev) return bad("null pointer (g, f_in_dev and f_out_dev are required)");
  if (nx < 1 || ny < 1 || nz < 5) return bad("need nx, ny >= 1 and nz >= 5 (three fluid layers for the plane ring)");
  if (precision < NH_FP64_SHIFTED || precision > NH_FP64_UNSHIFTED) return bad("precision must be 0..3");
  if (!(tau > 0.5) || !std::isfinite(tau)) return bad("tau must be > 0.5");
  if (!std::isfinite(g[0]) || !std::isfinite(g[1]) || !std::isfinite(g[2])) return bad("g must be finite");
  if (!(nx == 64 || nx == 128 || nx % 256 == 0)) return bad("nx must be 64, 128 or a multiple of 256 (pieces of 256 cells)");
  const double cells = (double)nx * ny * nz;
  if (cells * 19.0 >= 2147483648.0) return bad("grid too large: 19*nx*ny*nz must stay below 2^31");
  const size_t word = (precision == NH_FP32_SHIFTED || precision == NH_FP32_UNSHIFTED) ? 4 : 8;
  const size_t field_bytes = (size_t)19 * nx * ny * nz * word;

  // pieces of 256 cells on a ring plane of ny + 2 rows (one strip): whole rows per piece, or whole pieces per row
  Plan P;
  const unsigned pc = NT * U, rows = (unsigned)ny + 2;
  unsigned spr;
  if (pc % (unsigned)nx == 0) {
    P.rows_per_piece = pc / nx; spr = nx / (32u * U); P.ppr = 1;
    P.cps = (rows + P.rows_per_piece - 1) / P.rows_per_piece;
    P.pieces2 = ((unsigned)ny + P.rows_per_piece - 1) / P.rows_per_piece;
  } else {
    P.rows_per_piece = 1; spr = NT / 32; P.ppr = nx / pc;
    P.cps = rows * P.ppr;
    P.pieces2 = (unsigned)ny * P.ppr;
  }
  P.spr_shift = 0;
  while ((1u << P.spr_shift) < spr) ++P.spr_shift;
  P.nzf = nz - 2;
  P.order_len = 2u * (unsigned)P.nzf;
  P.flag_words = (size_t)P.nzf * P.cps;
  const size_t ctrl_words = HEADER_WORDS + nh::WAVE_MAX_STRIPS + 2 * P.flag_words + (P.order_len + 1) / 2;
  P.ctrl_bytes = (ctrl_words * 8 + ALIGN - 1) / ALIGN * ALIGN;
  P.plane_bytes = (size_t)19 * nx * rows * word;
  // ring of up to eight planes with the first phase four planes ahead (the handle path's defaults), fewer if they do not fit
  P.R = P.nzf < 8 ? P.nzf : 8;
  while (P.R >= 3 && P.ctrl_bytes + (size_t)P.R * P.plane_bytes > (size_t)NH_NOALLOC_SCRATCH_BYTES) --P.R;
  if (P.R < 3) {
    char msg[256];
    std::snprintf(msg, sizeof msg,
                  "lattice %dx%dx%d beyond the static scratch: needs %zu bytes (control block %zu + 3 ring planes of %zu), "
                  "the library holds %u; use nh_init_lattice with your own workspace",
                  nx, ny, nz, P.ctrl_bytes + 3 * P.plane_bytes, P.ctrl_bytes, P.plane_bytes, (unsigned)NH_NOALLOC_SCRATCH_BYTES);
    return bad(msg);
  }
  P.D = P.R - 2 < 4 ? P.R - 2 : 4;
  if ((unsigned long long)P.order_len * P.cps >= 2147483648ull) return bad("grid too large: too many work units");

  {
    const char* a = (const char*)f_in_dev;
    const char* b = (const char*)f_out_dev;
    if (a < b + field_bytes && b < a + field_bytes) return bad("f_in_dev and f_out_dev overlap");
  }
  unsigned char* scratch = nullptr;
  { const int rc = scratch_of_current_device(&scratch); if (rc) return rc; }
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  switch (precision) {
    case NH_FP64_SHIFTED: return run<double, true>(nx, ny, nz, tau, g, f_in_dev, F_lc_dev, f_out_dev, stream, scratch, P);
    case NH_FP32_SHIFTED: return run<float, true>(nx, ny, nz, tau, g, f_in_dev, F_lc_dev, f_out_dev, stream, scratch, P);
    case NH_FP32_UNSHIFTED: return run<float, false>(nx, ny, nz, tau, g, f_in_dev, F_lc_dev, f_out_dev, stream, scratch, P);
    default: return run<double, false>(nx, ny, nz, tau, g, f_in_dev, F_lc_dev, f_out_dev, stream, scratch, P);
  }
}
