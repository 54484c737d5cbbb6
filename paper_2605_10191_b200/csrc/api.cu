// Error reporting, handle lifetime and the CSR wrapper entry points of libpolfed.
#include <mutex>
#include <new>

#include "common.cuh"
#include "packed.cuh"

namespace polfed {

static thread_local std::string g_error;

void set_error(const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_error = buf;
}

int fail(int code, const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_error = buf;
  return code;
}

namespace {
constexpr int kMaxDev = 64;
std::mutex g_pool_mu;
cudaMemPool_t g_pools[kMaxDev] = {};
}  // namespace

cudaError_t scratch_alloc(void** p, size_t bytes, cudaStream_t st) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
  cudaMemPool_t pool;
  {
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (!g_pools[dev]) {
      cudaMemPoolProps props{};
      props.allocType = cudaMemAllocationTypePinned;
      props.handleTypes = cudaMemHandleTypeNone;
      props.location.type = cudaMemLocationTypeDevice;
      props.location.id = dev;
      e = cudaMemPoolCreate(&g_pools[dev], &props);
      if (e != cudaSuccess) return e;
      unsigned long long keep = ~0ull;
      e = cudaMemPoolSetAttribute(g_pools[dev], cudaMemPoolAttrReleaseThreshold, &keep);
      if (e != cudaSuccess) return e;
    }
    pool = g_pools[dev];
  }
  return cudaMallocFromPoolAsync(p, bytes ? bytes : 1, pool, st);
}

}  // namespace polfed

using polfed::fail;

extern "C" {

const char* polfed_last_error(void) { return polfed::g_error.c_str(); }

int polfed_release_scratch(void) {
  int dev = 0;
  POLFED_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= polfed::kMaxDev) return POLFED_OK;
  cudaMemPool_t pool;
  {
    std::lock_guard<std::mutex> lock(polfed::g_pool_mu);
    pool = polfed::g_pools[dev];
  }
  if (!pool) return POLFED_OK;
  POLFED_CUDA(cudaDeviceSynchronize());
  POLFED_CUDA(cudaMemPoolTrimTo(pool, 0));
  return POLFED_OK;
}

int polfed_version(void) { return 100; }  // 0.1.0

int polfed_ham_from_csr_ex(int64_t n, int64_t nnz, const int32_t* d_row_ptr, const int32_t* d_col,
                           const double* d_val, unsigned flags, void* stream, polfed_ham** out) {
  if (!out) return fail(POLFED_EINVAL, "polfed_ham_from_csr: out is NULL");
  *out = nullptr;
  if (n < 0 || nnz < 0) return fail(POLFED_EINVAL, "polfed_ham_from_csr: negative size");
  if (flags & ~(unsigned)POLFED_HAM_NO_SNAPSHOT)
    return fail(POLFED_EINVAL, "polfed_ham_from_csr_ex: unknown flag bits 0x%x", flags);
  if (n >= (int64_t(1) << 31) || nnz >= (int64_t(1) << 31))
    return fail(POLFED_ERANGE, "polfed_ham_from_csr: n and nnz must fit int32 indices");
  if (!d_row_ptr || (nnz > 0 && (!d_col || !d_val)))
    return fail(POLFED_EINVAL, "polfed_ham_from_csr: NULL array");
  if (!polfed::aligned16(d_val) || (reinterpret_cast<uintptr_t>(d_col) & 3u))
    return fail(POLFED_EINVAL, "polfed_ham_from_csr: misaligned array");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  polfed_ham* h = new (std::nothrow) polfed_ham;
  if (!h) return fail(POLFED_ENOMEM, "polfed_ham_from_csr: host allocation failed");
  h->n = n;
  h->nnz = nnz;
  h->d_row_ptr = d_row_ptr;
  h->d_col = d_col;
  h->d_val = d_val;
  h->owns = false;
  int dev = 0, sms = 148;
  if (cudaGetDevice(&dev) == cudaSuccess)
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  h->sm_count = sms > 0 ? sms : 148;
  cudaGetLastError();
  if (n <= 262144) {  // only the persistent small-matrix filter asks for it
    int rc = polfed::csr_max_row_len(n, d_row_ptr, &h->max_row_len, st);
    if (rc) {
      delete h;
      return rc;
    }
  }
  if (!(flags & POLFED_HAM_NO_SNAPSHOT)) {
    // the packed form of the same matrix, when its off-diagonal values are few (packed.cuh)
    int rc = polfed::build_packed_plan(h, st, &h->packed);
    if (rc) {
      delete h;
      return rc;
    }
  }
  *out = h;
  return POLFED_OK;
}

int polfed_ham_from_csr(int64_t n, int64_t nnz, const int32_t* d_row_ptr, const int32_t* d_col,
                        const double* d_val, polfed_ham** out) {
  return polfed_ham_from_csr_ex(n, nnz, d_row_ptr, d_col, d_val, 0u, nullptr, out);
}

int polfed_ham_destroy(polfed_ham* ham) {
  if (!ham) return POLFED_OK;
  polfed::destroy_tiled_plan(ham->tiled);
  polfed::destroy_flip_plan(ham->flip);
  polfed::destroy_packed_plan(ham->packed);
  if (ham->owns) {
    cudaFree(const_cast<int32_t*>(ham->d_row_ptr));
    cudaFree(const_cast<int32_t*>(ham->d_col));
    cudaFree(const_cast<double*>(ham->d_val));
  }
  delete ham;
  return POLFED_OK;
}

int polfed_ham_csr(const polfed_ham* ham, int64_t* n, int64_t* nnz, const int32_t** d_row_ptr,
                   const int32_t** d_col, const double** d_val) {
  if (!ham) return fail(POLFED_EINVAL, "polfed_ham_csr: ham is NULL");
  if (n) *n = ham->n;
  if (nnz) *nnz = ham->nnz;
  if (d_row_ptr) *d_row_ptr = ham->d_row_ptr;
  if (d_col) *d_col = ham->d_col;
  if (d_val) *d_val = ham->d_val;
  return POLFED_OK;
}

}  // extern "C"
