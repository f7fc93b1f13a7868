// ltv_scan_system_response_tube_static: the system response + tube call (eq.(12c), :147 eq.(12e)) for callers that
// cannot allocate device memory at all - code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
// The regular call takes its scratch (the per-(block, n-tile) tube partial sums `part`) as a caller-provided workspace; this
// variant keeps that scratch in a file-scope device array of a fixed, modest size, so the caller passes inputs and outputs
// only and the library calls no cudaMalloc / cudaFree / allocating routine on the way.
//
// The array lives in every CUDA context that loads the library, from load until exit (kStaticScratchBytes per GPU).  In host
// code its NAME is a host-side stand-in, not a device address: the address is fetched with cudaGetSymbolAddress, in this file,
// once per device, with that device current, and the pointer - not the name - goes to the kernels.  Every call on a device
// shares the one array, and it keeps the previous call's contents: the kernels of this call write every partial sum they later
// read (level 0 and the combine levels cover all blocks and n-tiles before the finalise kernel runs), so nothing has to start
// at zero and nothing is cleared.  Two calls that overlap on the GPU (different streams, or different host threads without
// stream ordering between them) RACE on the array; calls on one stream are ordered and safe.
#include <mutex>

#include "../../include/ltv_scan.h"
#include "ltv_internal.h"

namespace ltv {

namespace {

constexpr size_t kStaticScratchBytes = 32u << 20;   // 32 MiB: BASELINE.json configs[0] whole; about 27 items of configs[1], 6 of configs[2], 1 of configs[3]
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_scratch_mu;
void* g_scratch_ptr[kMaxDevices] = {};   // device address of g_static_scratch in the context of device i (nullptr: not asked yet)

// device address of the scratch array on the CURRENT device (looked up once per device)
cudaError_t static_scratch(void** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_scratch_mu);
  if (g_scratch_ptr[dev] == nullptr) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);   // the symbol of THIS translation unit, for the current device
    if (e != cudaSuccess) return e;
    if (p == nullptr) return cudaErrorInvalidSymbol;
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return cudaSuccess;
}

bool misaligned16(const void* p) { return p && (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

}  // namespace

}  // namespace ltv

using namespace ltv;

extern "C" {

size_t ltv_static_scratch_bytes(void) { return kStaticScratchBytes; }

int ltv_scan_system_response_tube_static(const float* A, const float* w, float* phi_out, float* r_out, int batch, int T,
                                         int n, unsigned flags, void* cuda_stream) {
  if (!A || !w || !r_out) return LTV_ERR_NULL_PTR;
  if (T > 1 && !phi_out) return LTV_ERR_NULL_PTR;
  if (batch < 1 || T < 1 || n < 1) return LTV_ERR_BAD_DIM;
  if ((flags & ~static_cast<unsigned>(LTV_TUBE_ROW_2NORM)) != 0) return LTV_ERR_BAD_DIM;
  if (n % 4 != 0 || n > 8192) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (static_cast<long long>(batch) * T * n >= (1ll << 31) ||
      static_cast<long long>(batch) * T * (T - 1) / 2 * n >= (1ll << 31))
    return LTV_ERR_UNSUPPORTED_SHAPE;
  // the scratch this problem needs = exactly what the regular call asks its caller for
  if (phi_workspace_bytes(batch, T, n, n) > kStaticScratchBytes) return LTV_ERR_STATIC_SCRATCH_LIMIT;
  if (misaligned16(A) || misaligned16(w) || misaligned16(phi_out) || misaligned16(r_out)) return LTV_ERR_ALIGNMENT;
  int dev = 0, major = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return report_cuda_error(e);
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) return report_cuda_error(e);
  if (major != 10) return LTV_ERR_ARCH;
  void* scratch = nullptr;
  e = static_scratch(&scratch);
  if (e != cudaSuccess) return report_cuda_error(e);
  PhiArgs a{A, w, phi_out, r_out, static_cast<float*>(scratch), batch, T, n, n, (flags & LTV_TUBE_ROW_2NORM) ? 1 : 0};
  unsigned long long l = 0;
  e = launch_phi_tube(a, static_cast<cudaStream_t>(cuda_stream), &l);   // the same kernels as the regular call
  count_launches(l);
  return e == cudaSuccess ? LTV_OK : report_cuda_error(e);
}

}  // extern "C"
