// er_api.cu -- status strings, size queries and device checks of the C ABI (include/er.h).
#include "er_common.cuh"

namespace er {
static thread_local int g_last_cuda_error = 0;
void set_last_cuda_error(int e) { g_last_cuda_error = e; }

int check_arch() {
  int dev = 0;
  ER_CUDA_TRY(cudaGetDevice(&dev));
  int major = 0;
  ER_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  return major == 10 ? ER_OK : ER_ERR_ARCH;
}

int current_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    (void)cudaGetLastError();
    return 0;
  }
  return dev;
}

// Per-device cache (a racing first call from two host threads writes the same value twice).
int sm_count() {
  static int cached[kMaxDevices] = {};
  const int dev = current_device();
  if (dev >= 0 && dev < kMaxDevices && cached[dev]) return cached[dev];
  int n = 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
    (void)cudaGetLastError();
    return 148;
  }
  if (dev >= 0 && dev < kMaxDevices) cached[dev] = n;
  return n;
}
}  // namespace er

extern "C" {

const char* er_status_str(int status) {
  switch (status) {
    case ER_OK: return "ER_OK";
    case ER_ERR_NULL: return "ER_ERR_NULL: a required pointer is NULL";
    case ER_ERR_SHAPE: return "ER_ERR_SHAPE: a size is outside the supported range";
    case ER_ERR_ALIGN: return "ER_ERR_ALIGN: pointer or leading dimension misaligned";
    case ER_ERR_DTYPE: return "ER_ERR_DTYPE: unsupported dtype / input form";
    case ER_ERR_WORKSPACE: return "ER_ERR_WORKSPACE: workspace missing or too small";
    case ER_ERR_ARCH: return "ER_ERR_ARCH: device is not sm_100 (no fallback path exists)";
    case ER_ERR_CUDA: return "ER_ERR_CUDA: CUDA call failed (see er_last_cuda_error)";
    default: return "ER_ERR_UNKNOWN";
  }
}

int er_last_cuda_error(void) { return er::g_last_cuda_error; }
int er_abi_version(void) { return ER_ABI_VERSION; }

size_t er_packed_bytes(int64_t N, int64_t K) {
  if (N < 128 || N % 128 != 0 || K < ER_GROUP || K % ER_GROUP != 0) return 0;
  return (size_t)N * (size_t)K / 2;
}

size_t er_scales_bytes(int64_t N, int64_t K, int group) {
  if (group != ER_GROUP || N < 128 || N % 128 != 0 || K < ER_GROUP || K % ER_GROUP != 0) return 0;
  return (size_t)(K / group) * (size_t)N * 2;
}

}  // extern "C"
