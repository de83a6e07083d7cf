// pibar.cu -- PI-BAR free-energy estimator (Eq. 27-28):
//   dF_AB = C + (1/beta) ln( <f(U_A - U_B + C)>_B / <f(U_B - U_A - C)>_A ),  C = dF_AB + (1/beta) ln(n_B/n_A),
//   f(x) = 1 / (1 + exp(beta x)), solved by fixed-point iteration from dF = 0 (reading G26).
// One cooperative kernel runs the whole iteration: every CTA sums the Fermi functions of its slice of
// the two stored series in a fixed order, the per-CTA partial sums meet in global memory, a grid-wide
// barrier, then every thread adds the partials in the same order, so all of them carry the same dF and
// leave the loop together.  The result does not depend on scheduling (no atomics).
#include <cooperative_groups.h>
#include <math.h>

#include <mutex>
#include <string>

#include "qhp_internal.cuh"

namespace cg = cooperative_groups;

#define PIBAR_THREADS 256

__global__ void __launch_bounds__(PIBAR_THREADS) k_pibar(const double *__restrict__ wA, long long nA,
                                                         const double *__restrict__ wB, long long nB, double beta,
                                                         int max_iter, double tol, double *part, double *out) {
  cg::grid_group grid = cg::this_grid();
  __shared__ double red[2][PIBAR_THREADS / 32];
  const int G = gridDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long gt = (long long)blockIdx.x * blockDim.x + tid, nth = (long long)G * blockDim.x;
  const double shift = log((double)nB / (double)nA) / beta;
  double dF = 0.0;
  int it = 0;
  while (it < max_iter) {
    const double C = dF + shift;                                                    // Eq. 28
    double sA = 0.0, sB = 0.0;
    for (long long i = gt; i < nA; i += nth) sA += 1.0 / (1.0 + exp(beta * (wA[i] - C)));   // f(U_B - U_A - C) on A
    for (long long j = gt; j < nB; j += nth) sB += 1.0 / (1.0 + exp(beta * (wB[j] + C)));   // f(U_A - U_B + C) on B
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      sA += __shfl_xor_sync(0xffffffffu, sA, o);
      sB += __shfl_xor_sync(0xffffffffu, sB, o);
    }
    if (lane == 0) { red[0][warp] = sA; red[1][warp] = sB; }
    __syncthreads();
    double *buf = part + (size_t)(it & 1) * 2 * G;          // two buffers: a CTA may be one iteration ahead
    if (tid == 0) {
      double a = 0.0, b = 0.0;
      for (int w = 0; w < PIBAR_THREADS / 32; ++w) { a += red[0][w]; b += red[1][w]; }
      buf[blockIdx.x] = a; buf[G + blockIdx.x] = b;
    }
    grid.sync();
    double tA = 0.0, tB = 0.0;
    for (int b = 0; b < G; ++b) { tA += __ldcg(buf + b); tB += __ldcg(buf + G + b); }
    const double dFn = C + log((tB / (double)nB) / (tA / (double)nA)) / beta;       // Eq. 27
    const double change = fabs(dFn - dF);
    dF = dFn;
    ++it;
    if (change <= tol) break;                                // identical on every thread of the grid
  }
  if (gt == 0) { out[0] = dF; out[1] = (double)it; }
}

extern "C" int qhp_pibar(const double *wA, int64_t nA, const double *wB, int64_t nB, double beta, int max_iter,
                         double tol, void *cuda_stream, double *dF_host, int *iters_host) {
  if (!wA || !wB || !dF_host || nA < 1 || nB < 1 || !(beta > 0) || max_iter < 1 || !(tol >= 0)) return QHP_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, coop = 0, sms = 0, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return QHP_ECUDA;
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_pibar, PIBAR_THREADS, 0) != cudaSuccess || per_sm < 1)
    return QHP_ECUDA;
  const long long n = nA > nB ? nA : nB;
  long long want = (n + PIBAR_THREADS - 1) / PIBAR_THREADS;
  int G = (int)(want < (long long)sms ? want : (long long)sms);      // one CTA per SM is plenty for a reduction
  double *scratch = nullptr;
  if (cudaMalloc(&scratch, sizeof(double) * (4 * (size_t)G + 2)) != cudaSuccess) return QHP_ENOMEM;
  double *part = scratch, *out = scratch + 4 * (size_t)G;
  long long a_n = nA, b_n = nB;
  void *args[] = {&wA, &a_n, &wB, &b_n, &beta, &max_iter, &tol, &part, &out};
  cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_pibar, dim3(G), dim3(PIBAR_THREADS), args, 0, st);
  double host[2] = {0.0, 0.0};
  if (e == cudaSuccess) e = cudaMemcpyAsync(host, out, sizeof(host), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(scratch);
  if (e != cudaSuccess) return QHP_ECUDA;
  *dF_host = host[0];
  if (iters_host) *iters_host = (int)host[1];
  return QHP_OK;
}

// ---------------------------------------------------------------------------------------------
// qhp_pibar_noalloc: the same kernel with its partial sums in a static device array (include/qhp.h).
// ---------------------------------------------------------------------------------------------
// File-scope scratch: 4 * MAX_CTAS doubles = 16 KiB on every GPU that loads the library.  In HOST code this
// name is only the host-side stand-in of the symbol, never a device address: the address the kernel gets is
// resolved per device by cudaGetSymbolAddress below.
static __device__ __align__(256) double pibar_scratch[4 * QHP_PIBAR_NOALLOC_MAX_CTAS];
static_assert(sizeof(double) * 4 * QHP_PIBAR_NOALLOC_MAX_CTAS == QHP_PIBAR_NOALLOC_SCRATCH_BYTES, "scratch size of include/qhp.h");

#define PIBAR_MAX_DEVICES 64
struct PibarDevice {
  bool ready = false;
  double *scratch = nullptr;   // device address of pibar_scratch on this device
  int sms = 0;
};
static PibarDevice g_pibar_dev[PIBAR_MAX_DEVICES];
static std::mutex g_pibar_mu;

// once per device, with that device current (the caller's current device is the one the launch goes to)
static int pibar_noalloc_setup(int dev, PibarDevice *out) {
  std::lock_guard<std::mutex> lock(g_pibar_mu);
  PibarDevice &d = g_pibar_dev[dev];
  if (!d.ready) {
    int coop = 0, per_sm = 0;
    void *ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, pibar_scratch);
    if (e != cudaSuccess || !ptr) {
      qhp_global_error((std::string("qhp_pibar_noalloc: cudaGetSymbolAddress(pibar_scratch): ") + cudaGetErrorString(e)).c_str());
      return QHP_ECUDA;
    }
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || !coop ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_pibar, PIBAR_THREADS, 0) != cudaSuccess || per_sm < 1) {
      qhp_global_error("qhp_pibar_noalloc: the device cannot launch the cooperative kernel");
      return QHP_ECUDA;
    }
    d.scratch = static_cast<double *>(ptr);
    d.ready = true;
  }
  *out = d;
  return QHP_OK;
}

extern "C" int qhp_pibar_noalloc(const double *wA, int64_t nA, const double *wB, int64_t nB, double beta, int max_iter,
                                 double tol, void *cuda_stream, double *out_dev) {
  if (!wA || !wB || !out_dev || nA < 1 || nB < 1 || !(beta > 0) || max_iter < 1 || !(tol >= 0)) {
    qhp_global_error("qhp_pibar_noalloc: bad argument (NULL pointer, empty series, beta <= 0, max_iter < 1 or tol < 0)");
    return QHP_EINVAL;
  }
  if (nA > QHP_PIBAR_NOALLOC_MAX_N || nB > QHP_PIBAR_NOALLOC_MAX_N) {
    qhp_global_error(("qhp_pibar_noalloc: series of " + std::to_string((long long)(nA > nB ? nA : nB)) +
                      " samples exceeds QHP_PIBAR_NOALLOC_MAX_N = " + std::to_string((long long)QHP_PIBAR_NOALLOC_MAX_N) +
                      " (static scratch, no allocation): use qhp_pibar").c_str());
    return QHP_EINVAL;
  }
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= PIBAR_MAX_DEVICES) {
    qhp_global_error("qhp_pibar_noalloc: no current CUDA device (or ordinal >= 64)");
    return QHP_ECUDA;
  }
  PibarDevice d;
  const int rc = pibar_noalloc_setup(dev, &d);
  if (rc) return rc;
  // the grid of qhp_pibar: same slices, same summation order, same result
  const long long n = nA > nB ? nA : nB;
  const long long want = (n + PIBAR_THREADS - 1) / PIBAR_THREADS;
  const int G = (int)(want < (long long)d.sms ? want : (long long)d.sms);
  if (G > QHP_PIBAR_NOALLOC_MAX_CTAS) {
    qhp_global_error(("qhp_pibar_noalloc: a grid of " + std::to_string(G) + " CTAs exceeds QHP_PIBAR_NOALLOC_MAX_CTAS = " +
                      std::to_string(QHP_PIBAR_NOALLOC_MAX_CTAS) + " (static scratch): use qhp_pibar").c_str());
    return QHP_EINVAL;
  }
  double *part = d.scratch;     // [2 buffers][2 series][G]; every entry read in an iteration is written in it first
  long long a_n = nA, b_n = nB;
  void *args[] = {&wA, &a_n, &wB, &b_n, &beta, &max_iter, &tol, &part, &out_dev};
  const cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_pibar, dim3(G), dim3(PIBAR_THREADS), args, 0,
                                                    (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) {
    qhp_global_error((std::string("qhp_pibar_noalloc: launch: ") + cudaGetErrorString(e)).c_str());
    return QHP_ECUDA;
  }
  return QHP_OK;
}
