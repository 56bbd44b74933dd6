// mcdc_noalloc.cu — mcdc_batch_stats_noalloc (include/mcdc.h): the batch close-out (SURVEY §8(a) row A14,
// DESIGN.md §3 C.9) and the mean / standard error of mcdc_tally_read(0 | 1) for callers that must not allocate
// device memory (CUDA graph capture, serving loops).  The launches are the ones of the workspace path — one
// k_closeout per batch folding into the running sums (sum x, sum x^2), then k_tally_stats — but the running sums
// live in a file-scope device array of fixed size instead of the caller's workspace.  Included at the end of
// mcdc_api.cu (same translation unit: the array, the address look-up and the launches see one another).
//
// The array exists once per device that loads the library, until the process exits.  Every call on a device
// shares it: calls that overlap on the GPU (different streams, or threads) race on it; a call leaves its sums
// behind, the next call's first close-out overwrites them (first = 1: write, not add), so nothing has to be
// cleared in between.

namespace mcdc {

constexpr size_t NOALLOC_MAX_BINS = MCDC_NOALLOC_MAX_BINS;
// [0, MAX) sum x, [MAX, 2 MAX) sum x^2: 16 MiB
static __device__ __align__(256) double g_noalloc_sums[2 * NOALLOC_MAX_BINS];

}  // namespace mcdc

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mu;
double *g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {nullptr};   // device address of g_noalloc_sums, per device
int g_noalloc_sms[NOALLOC_MAX_DEVICES] = {0};

// In host code `g_noalloc_sums` is only a handle of the symbol: the device address comes from
// cudaGetSymbolAddress, once per device, with that device current.
mcdc_status noalloc_setup(double **sums, int *sm_count)
{
  int dev = -1;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(MCDC_ECUDA, "device ordinal %d outside [0, %d)", dev, NOALLOC_MAX_DEVICES);
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    double *ptr = nullptr;
    CU(cudaGetSymbolAddress((void **)&ptr, mcdc::g_noalloc_sums));
    if (!ptr) return fail(MCDC_ECUDA, "cudaGetSymbolAddress returned a null address");
    int sms = 0;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    g_noalloc_sms[dev] = sms > 0 ? sms : 1;
    g_noalloc_ptr[dev] = ptr;
  }
  *sums = g_noalloc_ptr[dev];
  *sm_count = g_noalloc_sms[dev];
  return MCDC_OK;
}

}  // namespace

extern "C" mcdc_status mcdc_batch_stats_noalloc(const double *batches_dev, uint32_t n_batch, size_t n,
                                                double n_hist_per_batch, double *mean_dev, double *stderr_dev,
                                                void *cuda_stream)
{
  if (!batches_dev || !mean_dev) return fail(MCDC_EINVAL, "null argument");
  if (n_batch < 1 || n < 1) return fail(MCDC_EINVAL, "n_batch >= 1 and n >= 1");
  if (n > NOALLOC_MAX_BINS)
    return fail(MCDC_EINVAL, "n = %zu bins exceeds MCDC_NOALLOC_MAX_BINS = %zu (the fixed scratch array): use mcdc_run + mcdc_tally_read",
                n, (size_t)NOALLOC_MAX_BINS);
  if (!(n_hist_per_batch > 0.0) || !std::isfinite(n_hist_per_batch)) return fail(MCDC_EINVAL, "n_hist_per_batch > 0");
  double *sum1 = nullptr;
  int sms = 1;
  const mcdc_status st = noalloc_setup(&sum1, &sms);
  if (st != MCDC_OK) return st;
  double *sum2 = sum1 + NOALLOC_MAX_BINS;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  uint64_t g = (n + BS - 1) / BS;
  if (g > (uint64_t)sms * 8) g = (uint64_t)sms * 8;
  for (uint32_t b = 0; b < n_batch; ++b)
    k_closeout<<<(uint32_t)g, BS, 0, s>>>(batches_dev + (size_t)b * n, sum1, sum2, n, b == 0 ? 1 : 0);
  k_tally_stats<<<(uint32_t)g, BS, 0, s>>>(sum1, sum2, mean_dev, n, (double)n_batch, n_hist_per_batch, 0);
  if (stderr_dev)
    k_tally_stats<<<(uint32_t)g, BS, 0, s>>>(sum1, sum2, stderr_dev, n, (double)n_batch, n_hist_per_batch, 1);
  CU(cudaPeekAtLastError());
  return MCDC_OK;
}
