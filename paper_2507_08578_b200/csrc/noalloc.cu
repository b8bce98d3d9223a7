// noalloc.cu -- dft_apply_vloc_noalloc: the local term hpsi = FFT^-1[ V_loc(r) FFT[psi] ] (PAPER.md :475; SURVEY.md 8(a)
// S3-S7, the five pruned FFT passes of fft.cu / fft2.cu, unchanged) for callers that cannot allocate: code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The pass-to-pass scratch of the five passes
// (T1 [nb][ncol][n1] and T2 [nb][nplane][n2][n1] complex, which dft_apply_h takes from a cudaMalloc'ed or caller-supplied
// workspace) lives HERE in a file-scope device array of DFT_NOALLOC_SCRATCH_BYTES (64 MiB, include/dft.h): every GPU
// that loads the library holds that much device memory until the process exits.  The entry point calls no cudaMalloc,
// cudaFree or allocating library routine; the bands are processed in chunks that fit the array, and a plan whose
// scratch for ONE band exceeds it (boxes above about 190^3) is refused with DFT_ERR_ALLOC.
//
// All calls, of all plans on one GPU, share the array: calls that overlap on the GPU (different streams, no event
// between them) race on it.  The array keeps the contents of the last call; nothing has to start at zero, because every
// element a pass reads was written by the pass before it in the same call (pass A writes whole x-lines of T1, pass B
// whole planes of T2).
//
// `g_noalloc_scratch` in HOST code is only a stand-in for the symbol, not a device address: the address the kernels get
// comes from cudaGetSymbolAddress, asked once per device with that device current (below).
#include <mutex>

#include "../../include/dft.h"
#include "internal.h"

namespace dftb200 {

static __device__ __align__(256) unsigned char g_noalloc_scratch[DFT_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
void *g_scratch_addr[NOALLOC_MAX_DEVICES] = {nullptr};   // device address of the array on each device, once known
std::mutex g_scratch_mutex;

// device address of the scratch array on the CURRENT device (set-up on the first call per device)
int noalloc_scratch(void **out) {
  int dev = -1;
  DFT_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { set_error("device ordinal %d outside 0..%d", dev, NOALLOC_MAX_DEVICES - 1); return DFT_ERR_UNSUPPORTED; }
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    void *ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
    if (e != cudaSuccess || !ptr) {
      cudaGetLastError();
      set_error("cudaGetSymbolAddress of the static scratch array failed on device %d: %s", dev, cudaGetErrorString(e));
      return DFT_ERR_CUDA;
    }
    if ((uintptr_t)ptr & 255) { set_error("static scratch array is not 256-byte aligned"); return DFT_ERR_CUDA; }
    g_scratch_addr[dev] = ptr;
  }
  *out = g_scratch_addr[dev];
  return DFT_OK;
}

}  // namespace
}  // namespace dftb200

using namespace dftb200;

extern "C" int dft_apply_vloc_noalloc(dft_plan *p, const double *psi, double *hpsi, int32_t nband, void *stream) {
  if (!p) { set_error("null plan"); return DFT_ERR_INVALID_ARG; }
  if (nband < 0) { set_error("nband = %d is negative", nband); return DFT_ERR_INVALID_ARG; }
  if (nband == 0 || p->mpw == 0 || p->nkpt == 0) return DFT_OK;
  if (!psi || !hpsi) { set_error("null psi/hpsi"); return DFT_ERR_INVALID_ARG; }
  if (((uintptr_t)psi & 15) || ((uintptr_t)hpsi & 15)) { set_error("psi/hpsi must be 16-byte aligned"); return DFT_ERR_INVALID_ARG; }
  if (!p->vloc_set) { set_error("dft_apply_vloc_noalloc called before dft_set_vloc"); return DFT_ERR_NOT_READY; }
  const int64_t per_band = fft_ws_bytes_per_band(p);
  if (per_band > (int64_t)DFT_NOALLOC_SCRATCH_BYTES) {
    set_error("dft_apply_vloc_noalloc: one band of this plan needs %lld bytes of pass-to-pass scratch, the static array holds %lld "
              "(use dft_apply_h with dft_set_workspace instead)", (long long)per_band, (long long)DFT_NOALLOC_SCRATCH_BYTES);
    return DFT_ERR_ALLOC;
  }
  void *ws = nullptr;
  int rc = noalloc_scratch(&ws);
  if (rc) return rc;
  int64_t fit = per_band > 0 ? (int64_t)DFT_NOALLOC_SCRATCH_BYTES / per_band : nband;
  const int chunk = (int)(fit < nband ? fit : nband);
  cudaStream_t st = (cudaStream_t)stream;
  const bool timing = p->timer.on;     // the per-phase timers create events: off for this call
  p->timer.on = false;
  p->last_launches = 0;
  const size_t band_stride = (size_t)p->mpw * 2;
  for (int ik = 0; ik < p->nkpt && rc == DFT_OK; ik++)
    for (int b0 = 0; b0 < nband && rc == DFT_OK; b0 += chunk) {
      const int nb = nband - b0 < chunk ? nband - b0 : chunk;
      const size_t off = ((size_t)ik * nband + b0) * band_stride;
      rc = fft_apply_vloc(p, ik, psi + off, hpsi + off, nb, ws, st, nullptr);
    }
  p->timer.on = timing;
  return rc;
}
