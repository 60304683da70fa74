// foldcp_trimul_static (include/foldcp_trimul.h): foldcp_trimul for callers that cannot allocate
// device memory -- the workspace (a | b | o | LayerNorm(z) statistics | tile counters) lives in a
// file-scope __device__ array of FOLDCP_STATIC_WORKSPACE_BYTES instead of caller-owned memory.
//
// In HOST code the array's name is the host-side shadow of the symbol, not a device address (a
// kernel handed &g_static_workspace faults, or -- where the GPU can reach host memory -- silently
// uses the wrong memory).  The device address is taken with cudaGetSymbolAddress, once per device,
// with that device current, and it is that pointer which goes to foldcp_trimul and on to the
// kernels.  Nothing here (nor in foldcp_trimul below it) calls cudaMalloc / cudaFree or an
// allocating library routine; the tile counters at the workspace's tail are zeroed by a memset
// node on the caller's stream at every call, everything else in the workspace is written before
// it is read.
#include <atomic>

#include "common.h"

namespace foldcp {
namespace {

// every GPU on which this library's module is loaded holds these bytes until the process exits
static __device__ __align__(256) unsigned char g_static_workspace[FOLDCP_STATIC_WORKSPACE_BYTES];

constexpr int kMaxDevices = 64;
std::atomic<void*> g_static_ptr[kMaxDevices];   // device address of the array, per device ordinal

// Device address of g_static_workspace on the CURRENT device.  Two threads racing through the
// set-up both obtain the same address: the double store is harmless.
int static_workspace(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return FOLDCP_ERR_CUDA;
  if (dev < 0 || dev >= kMaxDevices) return FOLDCP_ERR_UNSUPPORTED;
  void* p = g_static_ptr[dev].load(std::memory_order_acquire);
  if (p == nullptr) {
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_workspace);
    if (e != cudaSuccess || p == nullptr) return FOLDCP_ERR_CUDA;   // cudaGetLastError keeps `e`
    if ((reinterpret_cast<uintptr_t>(p) & 255u) != 0) return FOLDCP_ERR_ALIGNMENT;
    g_static_ptr[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return FOLDCP_OK;
}

}  // namespace
}  // namespace foldcp

extern "C" {

size_t foldcp_trimul_static_workspace_bytes(void) { return FOLDCP_STATIC_WORKSPACE_BYTES; }

int foldcp_trimul_static_max_n(int c_z, int c_hidden, int dtype) {
  // foldcp_trimul_workspace_bytes is monotone in N; bf16 mode accepts multiples of 8 only
  const int step = dtype == FOLDCP_BF16 ? 8 : 1;
  int best = 0;
  for (int n = step; n <= 4096; n += step) {
    const size_t need = foldcp_trimul_workspace_bytes(n, c_z, c_hidden, dtype);
    if (need == 0 || need > FOLDCP_STATIC_WORKSPACE_BYTES) break;
    best = n;
  }
  return best;
}

int foldcp_trimul_static(const void* z, const void* mask, const foldcp_trimul_params* params, int N,
                         int c_z, int c_hidden, int direction, void* out, void* stream) {
  // the struct is copied below: its size must be the one this library was built with
  if (!params || params->struct_size != sizeof(foldcp_trimul_params)) return FOLDCP_ERR_INVALID_ARG;
  if (N <= 0) return FOLDCP_ERR_INVALID_ARG;
  const size_t need = foldcp_trimul_workspace_bytes(N, c_z, c_hidden, params->dtype);
  // need == 0: unsupported shape / dtype -- foldcp_trimul below names the reason
  if (need > FOLDCP_STATIC_WORKSPACE_BYTES) return FOLDCP_ERR_STATIC_LIMIT;
  void* ws = nullptr;
  const int st = foldcp::static_workspace(&ws);
  if (st != FOLDCP_OK) return st;
  foldcp_trimul_params p = *params;
  p.workspace = ws;
  p.workspace_bytes = FOLDCP_STATIC_WORKSPACE_BYTES;
  return foldcp_trimul(z, mask, &p, N, c_z, c_hidden, direction, out, stream);
}

}  // extern "C"
