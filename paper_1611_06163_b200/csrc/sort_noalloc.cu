// sort_noalloc.cu — row a2 of SURVEY §8(a) (the stable LSD radix sort of (cell key, previous slot)
// "radix sort") for callers that cannot allocate: tdpd_sort_cells_noalloc.  The kernels are the ones of binning.cu
// (td_launch_sort); what differs is where their scratch lives.  In a simulation the digit histograms, the chunk totals
// and the second side of the ping-pong come out of the caller's workspace; here they sit in ONE file-scope device
// array of fixed size, so the entry point calls no cudaMalloc / cudaFree and no allocating library routine.
//   - The array costs TDPD_NOALLOC_SCRATCH_BYTES on every GPU that loads the library, until the process exits.
//   - Its device address is asked for once per device (cudaGetSymbolAddress with that device current); in host code
//     the array's name is only a stand-in of the symbol and is never handed to a kernel.
//   - Nothing in it must start at zero: every histogram entry and chunk total a call reads was written by that call
//     (k_sort_hist writes all 256 bins of every tile, k_sort_scan every chunk total), and the ping-pong side is filled
//     from the input before it is read.  The contents of the last call stay behind and are never read.
//   - Every call on a device shares the array: two calls whose kernels overlap on the GPU (different streams, or two
//     host threads) race.  Calls on one stream are ordered and safe.
#include <cstdio>
#include <mutex>

#include "../../include/tdpd.h"
#include "common.cuh"

namespace {
constexpr int64_t MAXN = TDPD_NOALLOC_MAX_N;
constexpr size_t SIDE_BYTES = (size_t)MAXN * sizeof(uint32_t);                 // one array of keys or of values
constexpr size_t HIST_BYTES = TDPD_NOALLOC_SCRATCH_BYTES - 2 * SIDE_BYTES;      // histograms + chunk totals
static_assert(SIDE_BYTES % 256 == 0 && HIST_BYTES >= 96 * 1024, "scratch layout");

// [keys of the scratch side][values of the scratch side][digit histograms, chunk totals]
static __device__ __align__(256) unsigned char g_sort_scratch[TDPD_NOALLOC_SCRATCH_BYTES];

constexpr int MAX_DEV = 64;
std::mutex g_mu;
unsigned char* g_scratch_of[MAX_DEV];  // device address of g_sort_scratch, by device ordinal (0 = not asked yet)
thread_local char g_msg[256] = "";

int fail(int code, const char* fmt, long long a = 0, long long b = 0) {
  snprintf(g_msg, sizeof g_msg, fmt, a, b);
  return code;
}

// device address of the scratch array on the current device
int scratch_address(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(TDPD_ECUDA, "cudaGetDevice failed (%lld)", (long long)e);
  if (dev < 0 || dev >= MAX_DEV) return fail(TDPD_EINVAL, "device ordinal %lld beyond the %lld this entry point keeps", dev, MAX_DEV);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_of[dev]) {
    unsigned char* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_sort_scratch);
    if (e != cudaSuccess || !p) return fail(TDPD_ECUDA, "cudaGetSymbolAddress of the sort scratch failed (%lld) on device %lld", (long long)e, dev);
    g_scratch_of[dev] = p;
  }
  *out = g_scratch_of[dev];
  return TDPD_OK;
}

__global__ void __launch_bounds__(256) k_iota(uint32_t* __restrict__ v, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) v[i] = (uint32_t)i;
}
}  // namespace

extern "C" int tdpd_noalloc_init(void) {
  unsigned char* p = nullptr;
  const int rc = scratch_address(&p);
  if (rc == TDPD_OK) g_msg[0] = 0;
  return rc;
}

extern "C" const char* tdpd_noalloc_last_error(void) { return g_msg; }

extern "C" int tdpd_sort_cells_noalloc(const uint32_t* d_keys, const uint32_t* d_vals, int64_t n, int32_t key_bits,
                                       uint32_t* d_keys_out, uint32_t* d_vals_out, void* stream) {
  if (n < 0) return fail(TDPD_EINVAL, "n = %lld is negative", n);
  if (n > MAXN)
    return fail(TDPD_EINVAL, "n = %lld exceeds TDPD_NOALLOC_MAX_N = %lld: the scratch of this entry point is a fixed device array; "
                             "sort larger systems inside a tdpd_sim (caller-provided workspace)", n, MAXN);
  if (key_bits < 1 || key_bits > 32) return fail(TDPD_EINVAL, "key_bits = %lld outside 1..32", key_bits);
  if (n == 0) { g_msg[0] = 0; return TDPD_OK; }
  if (!d_keys || !d_keys_out || !d_vals_out) return fail(TDPD_EINVAL, "d_keys, d_keys_out and d_vals_out must not be NULL");
  if (td_sort_scratch_bytes(n) > HIST_BYTES) return fail(TDPD_ENOMEM, "histograms of n = %lld do not fit the scratch (%lld bytes)", n, (long long)HIST_BYTES);
  unsigned char* base = nullptr;
  int rc = scratch_address(&base);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  uint32_t* const sk = (uint32_t*)base;
  uint32_t* const sv = (uint32_t*)(base + SIDE_BYTES);
  void* const hist = base + 2 * SIDE_BYTES;
  // The sort starts on side 0 and ends on side (passes & 1): the caller's output arrays take the side it ends on,
  // the scratch takes the other, so the result lands in place and needs no copy.
  const int so = td_sort_passes(key_bits) & 1;
  uint32_t* keys[2];
  uint32_t* vals[2];
  keys[so] = d_keys_out; vals[so] = d_vals_out;
  keys[so ^ 1] = sk; vals[so ^ 1] = sv;
  cudaError_t e = cudaSuccess;
  if (keys[0] != d_keys) e = cudaMemcpyAsync(keys[0], d_keys, (size_t)n * 4, cudaMemcpyDeviceToDevice, st);
  if (e == cudaSuccess) {
    if (d_vals) {
      if (vals[0] != d_vals) e = cudaMemcpyAsync(vals[0], d_vals, (size_t)n * 4, cudaMemcpyDeviceToDevice, st);
    } else {
      k_iota<<<(int)((n + 255) / 256), 256, 0, st>>>(vals[0], n);
    }
  }
  if (e != cudaSuccess) return fail(TDPD_ECUDA, "staging the input failed (%lld)", (long long)e);
  const int side = td_launch_sort(keys, vals, n, key_bits, hist, st, nullptr, nullptr);
  if (side != so) return fail(TDPD_ECUDA, "sort ended on side %lld, expected %lld", side, so);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(TDPD_ECUDA, "kernel launch failed (%lld)", (long long)e);
  g_msg[0] = 0;
  return TDPD_OK;
}
