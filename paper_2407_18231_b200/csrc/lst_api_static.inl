// lst_api_static.inl -- included by lst_api.cu (same translation unit as the array below): the slot-offset
// scan of the chain (lst_ingest.cuh, scan_body) as two stand-alone entry points.
//
//   lst_scan_counts         the chain's own kernel (k_scan), its ticket and tile status words taken from
//                           cudaMalloc for the duration of the call;
//   lst_scan_counts_static  the same tile loop with ticket and status words in g_scan_scratch, a fixed array
//                           that is part of the loaded library image: no allocation of any kind per call.
//
// Who needs the second one: code that runs where a device allocation is not allowed or not affordable --
// a trigger / reconstruction framework (PAPER.md:79 measures LST inside one) whose device memory belongs to
// the framework's pool and whose modules may not call cudaMalloc / cudaFree in the event loop, because both
// synchronise the whole device and stall every other stream; and callers that are inside a region where the
// runtime refuses to allocate at all.

namespace {

constexpr int kStaticScanTiles = LST_SCAN_STATIC_MAX_N / kScanTile + 2;
constexpr size_t kStaticScanHead = 256;  // the tile ticket lives in the first word; the status words start here
constexpr size_t kStaticScanBytes = kStaticScanHead + sizeof(unsigned long long) * kStaticScanTiles;

// The scratch of lst_scan_counts_static: about 128 KB, resident on every GPU that loads this library, until
// the process exits.  In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device
// address and must never be handed to a kernel.
static __device__ __align__(256) unsigned char g_scan_scratch[kStaticScanBytes];

// Variant of k_scan: identical tile loop; ticket and status words are offsets into one scratch block.
__global__ void __launch_bounds__(kBlock)
k_scan_static(const int* __restrict__ in, int* __restrict__ out, int n, unsigned char* scratch) {
  scan_body<kScanItems>(ScanJob{in, out, nullptr, 0, n, reinterpret_cast<int*>(scratch),
                                reinterpret_cast<unsigned long long*>(scratch + kStaticScanHead)});
}

// Per device: the device address of g_scan_scratch and the SM count, looked up once (first call on that device).
constexpr int kStaticMaxDevices = 64;
struct StaticScanDevice {
  unsigned char* scratch;
  int n_sm;
};
StaticScanDevice g_static_dev[kStaticMaxDevices];  // zero-initialised: scratch == nullptr means "not set up"
std::mutex g_static_mu;

int static_scan_setup(StaticScanDevice* out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) return LST_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (dev < kStaticMaxDevices && g_static_dev[dev].scratch) {
    *out = g_static_dev[dev];
    return LST_OK;
  }
  // `dev` is the current device: the address returned is the one of ITS copy of the array
  StaticScanDevice s{nullptr, 0};
  void* p = nullptr;
  if (cudaGetSymbolAddress(&p, g_scan_scratch) != cudaSuccess || !p) {
    cudaGetLastError();
    return LST_ERR_CUDA;
  }
  if (cudaDeviceGetAttribute(&s.n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || s.n_sm < 1) {
    cudaGetLastError();
    return LST_ERR_CUDA;
  }
  s.scratch = static_cast<unsigned char*>(p);
  if (dev < kStaticMaxDevices) g_static_dev[dev] = s;  // beyond the table: looked up again on every call
  *out = s;
  return LST_OK;
}

inline int scan_args_ok(const int32_t* counts, int32_t n, const int32_t* offsets) {
  if (n < 0 || !offsets || (n > 0 && !counts)) return LST_ERR_ARG;
  if (n > 0 && (reinterpret_cast<uintptr_t>(counts) & 15u)) return LST_ERR_ARG;  // 16-byte loads
  return LST_OK;
}

inline int scan_tiles(int n) { return n > 0 ? (n + kScanTile - 1) / kScanTile : 1; }

}  // namespace

extern "C" int lst_scan_counts(const int32_t* counts, int32_t n, int32_t* offsets, void* cuda_stream) {
  const int rc = scan_args_ok(counts, n, offsets);
  if (rc != LST_OK) return rc;
  int dev = 0, n_sm = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int tiles = scan_tiles(n);
  const size_t bytes = kStaticScanHead + sizeof(unsigned long long) * ((size_t)tiles + 2);
  unsigned char* scratch = nullptr;
  if (cudaMalloc(&scratch, bytes) != cudaSuccess) {
    cudaGetLastError();
    return LST_ERR_CUDA;
  }
  bool ok = cudaMemsetAsync(scratch, 0, bytes, st) == cudaSuccess;
  if (ok) {
    k_scan<<<tiles < 4 * n_sm ? tiles : 4 * n_sm, kBlock, 0, st>>>(
        counts, offsets, nullptr, 0, n, reinterpret_cast<int*>(scratch),
        reinterpret_cast<unsigned long long*>(scratch + kStaticScanHead));
    ok = cudaGetLastError() == cudaSuccess && cudaStreamSynchronize(st) == cudaSuccess;
  }
  cudaFree(scratch);
  return ok ? LST_OK : LST_ERR_CUDA;
}

extern "C" int lst_scan_counts_static(const int32_t* counts, int32_t n, int32_t* offsets, void* cuda_stream) {
  const int rc = scan_args_ok(counts, n, offsets);
  if (rc != LST_OK) return rc;
  if (n > LST_SCAN_STATIC_MAX_N) return LST_ERR_LIMIT;
  StaticScanDevice sd;
  const int sr = static_scan_setup(&sd);
  if (sr != LST_OK) return sr;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int tiles = scan_tiles(n);
  // The array still holds the ticket and the status words of whatever call used it last: the part this call
  // reads must be zero again ("no tile has published anything") before its kernel starts.
  CK(cudaMemsetAsync(sd.scratch, 0, kStaticScanHead + sizeof(unsigned long long) * (size_t)tiles, st));
  k_scan_static<<<tiles < 4 * sd.n_sm ? tiles : 4 * sd.n_sm, kBlock, 0, st>>>(counts, offsets, n, sd.scratch);
  CK(cudaGetLastError());
  return LST_OK;
}
