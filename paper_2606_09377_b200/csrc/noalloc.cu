// crown_gemm_noalloc -- the A.W contraction of Eq. 1 for callers that cannot allocate device
// memory (code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// crown_gemm needs the TF32 hi/lo limbs of both operands in caller-provided buffers (crown_split_tf32 writes them);
// here those limbs live in ONE file-scope device array of fixed size, so the entry point takes only the fp32 operands
// and the output.  It calls no cudaMalloc / cudaFree / allocating library routine and needs no crown_ctx (crown_init
// pins host memory); error text goes to a fixed thread-local buffer.
//
// The array is shared by every call in the process and keeps the last call's contents.  Both split kernels overwrite
// every limb the contraction then reads (rows beyond M / N are zero-filled by the TMA, not read from the array) and
// the contraction's first K panel stores D without reading it (later panels add into what the first one stored), so
// nothing has to start at zero and nothing is cleared.
// Two calls whose kernels overlap on the GPU (different streams, no dependency between them) RACE on the array.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/crownb200.h"
#include "kernels.h"

namespace {

constexpr size_t MAX_ELEMS = CROWN_GEMM_NOALLOC_MAX_ELEMS;   // M*K + N*K, each rounded up to 64 elements
// [hi limbs | lo limbs], each MAX_ELEMS floats: 2 * 2^21 * 4 B = 16 MiB on every GPU that loads the library
static __device__ __align__(256) float g_limbs[2 * MAX_ELEMS];

constexpr int MAX_DEVICES = 64;
struct PerDevice { float* limbs = nullptr; int num_sms = 0; };
PerDevice g_dev[MAX_DEVICES];
std::mutex g_mu;

thread_local char t_err[256] = "";

int fail(int code, const char* what, const char* detail = nullptr) {
  if (detail) snprintf(t_err, sizeof t_err, "crown_gemm_noalloc: %s: %s", what, detail);
  else snprintf(t_err, sizeof t_err, "crown_gemm_noalloc: %s", what);
  return code;
}

// Once per device, with that device current: in host code `g_limbs` is a host-side stand-in for the symbol, not a
// device address -- the address the kernels get comes from cudaGetSymbolAddress.
int setup_device(int dev, PerDevice* out) {
  std::lock_guard<std::mutex> lock(g_mu);
  PerDevice& pd = g_dev[dev];
  if (!pd.limbs) {
    float* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_limbs);
    if (e != cudaSuccess) return fail(CROWN_ECUDA, "cudaGetSymbolAddress", cudaGetErrorString(e));
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255) != 0) return fail(CROWN_ECUDA, "scratch symbol is not 256-byte aligned");
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess || sms <= 0) return fail(CROWN_ECUDA, "cudaDeviceGetAttribute", cudaGetErrorString(e));
    if (crownb200::gemm_tc_init_device() != 0) {        // opt-in shared memory size + resident CTA-pair count
      (void)cudaGetLastError();
      return fail(CROWN_ECUDA, "the tcgen05 contraction kernel cannot be configured on this device (sm_100a only)");
    }
    pd.num_sms = sms;
    pd.limbs = p;
  }
  *out = pd;
  return CROWN_OK;
}

inline size_t round64(size_t x) { return (x + 63) / 64 * 64; }

}  // namespace

extern "C" int crown_gemm_noalloc_max_elems(void) { return (int)MAX_ELEMS; }

extern "C" const char* crown_gemm_noalloc_error(void) { return t_err; }

extern "C" int crown_gemm_noalloc(int M, int N, int K, const float* A_dev, const float* W_dev, float* D_dev, void* stream) {
  t_err[0] = 0;
  if (M <= 0 || N <= 0 || K <= 0 || !A_dev || !W_dev || !D_dev) return fail(CROWN_EINVAL, "bad arguments (null pointer or size <= 0)");
  if (!crownb200::gemm_tc_supported(M, N, K))
    return fail(CROWN_EINVAL, "shape outside the tensor-core tile rules: need N >= 128, K >= 32, N % 4 == 0, K % 4 == 0");
  if ((reinterpret_cast<uintptr_t>(D_dev) & 15) != 0) return fail(CROWN_EINVAL, "D_dev must be 16-byte aligned");
  const size_t na = round64((size_t)M * (size_t)K), nw = round64((size_t)N * (size_t)K);
  if (na + nw > MAX_ELEMS) {
    char msg[160];
    snprintf(msg, sizeof msg, "M*K + N*K = %zu elements (each rounded up to 64) exceeds the static scratch of %zu; use crown_gemm with caller buffers",
             na + nw, MAX_ELEMS);
    return fail(CROWN_EINVAL, "problem too large", msg);
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(CROWN_ECUDA, "cudaGetDevice", cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(CROWN_EUNSUPPORTED, "device ordinal beyond 63");
  PerDevice pd;
  if (int rc = setup_device(dev, &pd)) return rc;

  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  float* A_hi = pd.limbs;
  float* Wt_hi = pd.limbs + na;
  float* A_lo = pd.limbs + MAX_ELEMS;
  float* Wt_lo = pd.limbs + MAX_ELEMS + na;
  crownb200::launch_split_tf32(A_dev, M, K, 0, A_hi, A_lo, s);          // A [M,K]   -> limbs [M,K]
  crownb200::launch_split_tf32(W_dev, K, N, 1, Wt_hi, Wt_lo, s);        // W [K,N]   -> limbs of W^T [N,K]
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(CROWN_ECUDA, "operand split launch", cudaGetErrorString(e));
  const char* why = nullptr;
  if (crownb200::launch_gemm_tc(A_hi, A_lo, Wt_hi, Wt_lo, D_dev, N, M, N, K, 0, pd.num_sms, s, &why))
    return fail(CROWN_ECUDA, "contraction launch", why ? why : "?");
  return CROWN_OK;
}
