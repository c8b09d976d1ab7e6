// Broyden's modified second method, Algorithm 3 of the paper, one GPU.
// (a6 of SURVEY.md 8(a).)  Steps are numbered as in the paper.  Readings R15-R19 of DESIGN.md:
// zeta in step 13, sliding window of `history` (v, w) pairs summed oldest first -- when the window is
// full the oldest pair leaves BEFORE steps 9-11, so that the new pair satisfies the secant equation
// G_{m+1} df_m = dx_m with G = zeta I + sum over the kept pairs (R17) --, d = 0 skips steps 9-13,
// eps_t = |f_t| / max(|x_in + x_out|, 1e-300); a non-finite residual gives eps_max = +infinity.
//
// The paper's atomics (steps 5, 6, 9, 14) are replaced by warp-shuffle + shared
// memory block reductions and a fixed-order second stage, so results are bit-reproducible.  All dot
// products of one iteration (V^T df, V^T f, df.df, df.f) come from ONE pass over the vectors: the new
// pair's k_m = v_m.f equals (df.f)/d, so steps 14-15 need no second reduction.
#include <math_constants.h>

#include <new>

#include "negf_internal.h"

namespace negf {
namespace {

constexpr int kChunk = 8;          // stored pairs handled per dots launch
constexpr int kThreads = 256;

struct Plan {              // device-resident ring-buffer state
  int n_stored;            // pairs stored before this step
  int head;                // slot of the oldest stored pair
  int m;                   // iteration counter of Alg.3
  int do_store;            // this step adds a pair (m > 0 and d != 0)
  int slot_new;            // slot the new pair goes to
  int evict;               // the window is full: the oldest pair is dropped before steps 9-11 (R17)
};

struct Dots {              // results of the reductions, device memory
  double d;                // ||df||^2          (steps 6, 8)
  double e;                // df . f
  double eps_max;          // steps 4-7
  double pad;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
// max that does not lose a non-finite residual: fmax drops NaN, and a caller looping on
// "eps_max >= 1e-5" would then declare convergence on a NaN state.  NaN and
// infinity both map to +infinity.
__device__ __forceinline__ double nan_max(double a, double b) {
  if (!(fabs(b) <= 1.79769313486231570e308)) b = CUDART_INF;
  return (a >= b) ? a : b;       // a is never NaN by construction
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = nan_max(v, __shfl_down_sync(0xffffffffu, v, o));
  return v;
}

// partial layout: part[block][2*kChunk + 3]
__global__ void __launch_bounds__(kThreads)
broyden_dots_kernel(const double* __restrict__ x_in, const double* __restrict__ x_out,
                    const double* __restrict__ f_old, const double* __restrict__ V, int64_t len,
                    int history, const Plan* __restrict__ plan, int chunk0, int first,
                    double* __restrict__ part) {
  __shared__ double sm[kThreads / 32][2 * kChunk + 3];
  const int n_stored = plan->n_stored, head = plan->head;
  const int nj = max(0, min(kChunk, n_stored - chunk0));
  double k1[kChunk], k2[kChunk];
#pragma unroll
  for (int j = 0; j < kChunk; ++j) k1[j] = k2[j] = 0.0;
  double d = 0.0, e = 0.0, em = 0.0;
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < len;
       t += (int64_t)gridDim.x * kThreads) {
    const double xi = x_in[t], xo = x_out[t];
    const double f = xi - xo;                                  // step 2
    const double df = f - f_old[t];                            // step 3
    if (first) {
      em = nan_max(em, fabs(f) / fmax(fabs(xi + xo), 1e-300)); // step 4
      d += df * df;                                            // step 6
      e += df * f;
    }
#pragma unroll
    for (int j = 0; j < kChunk; ++j) {
      if (j < nj) {
        const int slot = (head + chunk0 + j) % history;        // age order, oldest first
        const double v = V[(size_t)slot * len + t];
        k1[j] += v * df;                                       // step 9
        k2[j] += v * f;                                        // step 14
      }
    }
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < kChunk; ++j) {
    k1[j] = warp_sum(k1[j]);
    k2[j] = warp_sum(k2[j]);
  }
  d = warp_sum(d);
  e = warp_sum(e);
  em = warp_max(em);
  if (lane == 0) {
#pragma unroll
    for (int j = 0; j < kChunk; ++j) {
      sm[wid][j] = k1[j];
      sm[wid][kChunk + j] = k2[j];
    }
    sm[wid][2 * kChunk] = d;
    sm[wid][2 * kChunk + 1] = e;
    sm[wid][2 * kChunk + 2] = em;
  }
  __syncthreads();
  if (threadIdx.x < 2 * kChunk + 3) {
    double t = 0.0;
    if (threadIdx.x == 2 * kChunk + 2) {
      for (int w = 0; w < kThreads / 32; ++w) t = nan_max(t, sm[w][threadIdx.x]);
    } else {
      for (int w = 0; w < kThreads / 32; ++w) t += sm[w][threadIdx.x];
    }
    part[(size_t)blockIdx.x * (2 * kChunk + 3) + threadIdx.x] = t;
  }
}

// single block: fixed-order sum over the blocks' partials; the chunk's k1/k2 go to kbuf.
__global__ void broyden_finish_kernel(const double* __restrict__ part, int nblocks, int chunk0,
                                      int first, int last, int history, double* __restrict__ k1buf,
                                      double* __restrict__ k2buf, Dots* __restrict__ dots,
                                      Plan* __restrict__ plan) {
  const int q = threadIdx.x;
  if (q < 2 * kChunk + 3) {
    double t = 0.0;
    if (q == 2 * kChunk + 2) {
      for (int b = 0; b < nblocks; ++b) t = nan_max(t, part[(size_t)b * (2 * kChunk + 3) + q]);
    } else {
      for (int b = 0; b < nblocks; ++b) t += part[(size_t)b * (2 * kChunk + 3) + q];
    }
    if (q < kChunk) k1buf[chunk0 + q] = t;
    else if (q < 2 * kChunk) k2buf[chunk0 + q - kChunk] = t;
    else if (first) {
      if (q == 2 * kChunk) dots->d = t;
      else if (q == 2 * kChunk + 1) dots->e = t;
      else dots->eps_max = t;
    }
  }
  __syncthreads();
  if (last && q == 0) {
    const int store = (plan->m > 0 && dots->d != 0.0) ? 1 : 0;       // R18
    plan->do_store = store;
    if (store) {
      if (plan->n_stored < history) {
        plan->evict = 0;
        plan->slot_new = (plan->head + plan->n_stored) % history;
      } else {
        plan->evict = 1;                                              // R17
        plan->slot_new = plan->head;
      }
    } else {
      plan->evict = 0;
      plan->slot_new = 0;
    }
  }
}

__global__ void __launch_bounds__(kThreads)
broyden_update_kernel(double* __restrict__ x_in, const double* __restrict__ x_out,
                      double* __restrict__ f_old, double* __restrict__ x_old, double* __restrict__ V,
                      double* __restrict__ W, int64_t len, int history, double zeta,
                      const Plan* __restrict__ plan, const double* __restrict__ k1buf,
                      const double* __restrict__ k2buf, const Dots* __restrict__ dots) {
  const int n_stored = plan->n_stored, head = plan->head;
  const int store = plan->do_store, slot_new = plan->slot_new, evict = plan->evict;
  const double d = dots->d, e = dots->e;
  for (int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x; t < len;
       t += (int64_t)gridDim.x * kThreads) {
    const double xi = x_in[t];
    const double f = xi - x_out[t];
    const double df = f - f_old[t];
    double s2 = 0.0;
    double w_new = 0.0;
    if (store) {
      double s1 = 0.0;
      for (int j = evict; j < n_stored; ++j)                              // steps 10-11 (R17: kept pairs)
        s1 += W[(size_t)((head + j) % history) * len + t] * k1buf[j];
      w_new = -zeta * df + (xi - x_old[t]) - s1;                          // step 13 (R15)
    }
    for (int j = evict; j < n_stored; ++j)                                // steps 15-16
      s2 += W[(size_t)((head + j) % history) * len + t] * k2buf[j];
    if (store) {
      s2 += w_new * (e / d);                                              // k_m = v_m . f = (df.f)/d
      V[(size_t)slot_new * len + t] = df / d;                             // step 12
      W[(size_t)slot_new * len + t] = w_new;
    }
    x_old[t] = xi;                                                        // step 17
    f_old[t] = f;
    x_in[t] = xi - zeta * f - s2;                                         // step 18
  }
}

__global__ void broyden_advance_kernel(Plan* plan, int history) {          // step 19
  if (plan->do_store) {
    if (plan->evict) plan->head = (plan->head + 1) % history;
    else plan->n_stored += 1;
  }
  plan->m += 1;
}

}  // namespace
}  // namespace negf

using namespace negf;

struct broyden_handle {
  int64_t len;
  int history;
  double zeta;
  cudaStream_t stream;
  int nblocks;
  double *f_old, *x_old, *V, *W, *part, *k1buf, *k2buf;
  Dots* dots;
  Plan* plan;
  double* eps_pinned;
};

extern "C" negf_status broyden_reset(broyden_handle* h) {
  if (!h) { set_error("broyden_reset: null handle"); return NEGF_EINVAL; }
  NEGF_CUDA_TRY(cudaMemsetAsync(h->f_old, 0, sizeof(double) * h->len, h->stream));
  NEGF_CUDA_TRY(cudaMemsetAsync(h->x_old, 0, sizeof(double) * h->len, h->stream));
  NEGF_CUDA_TRY(cudaMemsetAsync(h->plan, 0, sizeof(Plan), h->stream));
  NEGF_CUDA_TRY(cudaMemsetAsync(h->dots, 0, sizeof(Dots), h->stream));
  return NEGF_OK;
}

extern "C" negf_status broyden_destroy(broyden_handle* h) {
  if (!h) return NEGF_OK;
  cudaFree(h->f_old); cudaFree(h->x_old); cudaFree(h->V); cudaFree(h->W); cudaFree(h->part);
  cudaFree(h->k1buf); cudaFree(h->k2buf); cudaFree(h->dots); cudaFree(h->plan);
  if (h->eps_pinned) cudaFreeHost(h->eps_pinned);
  delete h;
  return NEGF_OK;
}

extern "C" negf_status broyden_create(int64_t len, int32_t history, double zeta, void* cuda_stream,
                                      broyden_handle** out) {
  if (!out) { set_error("broyden_create: out is null"); return NEGF_EINVAL; }
  *out = nullptr;
  if (len < 1 || history < 1 || history > 4096 || !(zeta > 0.0)) {
    set_error("broyden_create: need len >= 1, 1 <= history <= 4096, zeta > 0");
    return NEGF_EINVAL;
  }
  broyden_handle* h = new (std::nothrow) broyden_handle();
  if (!h) { set_error("broyden_create: out of host memory"); return NEGF_ENOMEM; }
  h->len = len; h->history = history; h->zeta = zeta;
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  int64_t nb = (len + kThreads - 1) / kThreads;
  h->nblocks = (int)(nb < 1184 ? nb : 1184);        // 148 SMs x 8 resident blocks
  const int hpad = ((history + kChunk - 1) / kChunk) * kChunk;
  cudaError_t e = cudaSuccess;
  auto alloc = [&](void** p, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(p, bytes); };
  alloc((void**)&h->f_old, sizeof(double) * len);
  alloc((void**)&h->x_old, sizeof(double) * len);
  alloc((void**)&h->V, sizeof(double) * len * history);
  alloc((void**)&h->W, sizeof(double) * len * history);
  alloc((void**)&h->part, sizeof(double) * h->nblocks * (2 * kChunk + 3));
  alloc((void**)&h->k1buf, sizeof(double) * hpad);
  alloc((void**)&h->k2buf, sizeof(double) * hpad);
  alloc((void**)&h->dots, sizeof(Dots));
  alloc((void**)&h->plan, sizeof(Plan));
  if (e == cudaSuccess) e = cudaMallocHost((void**)&h->eps_pinned, sizeof(double));
  if (e != cudaSuccess) {
    set_error("broyden_create: allocation failed: %s", cudaGetErrorString(e));
    negf_status st = (e == cudaErrorMemoryAllocation) ? NEGF_ENOMEM : NEGF_ECUDA;
    broyden_destroy(h);
    return st;
  }
  negf_status st = broyden_reset(h);
  if (st != NEGF_OK) { broyden_destroy(h); return st; }
  *out = h;
  return NEGF_OK;
}

extern "C" negf_status broyden_step(broyden_handle* h, double* x_in_dev, const double* x_out_dev,
                                    double* eps_max_host) {
  if (!h || !x_in_dev || !x_out_dev) { set_error("broyden_step: null argument"); return NEGF_EINVAL; }
  const int nchunks = (h->history + kChunk - 1) / kChunk;
  // Pairs beyond n_stored contribute nothing, so all chunks can always be launched; the number of
  // stored pairs lives on the device (no host sync needed to know it).
  for (int c = 0; c < nchunks; ++c) {
    broyden_dots_kernel<<<h->nblocks, kThreads, 0, h->stream>>>(
        x_in_dev, x_out_dev, h->f_old, h->V, h->len, h->history, h->plan, c * kChunk, c == 0, h->part);
    broyden_finish_kernel<<<1, 32, 0, h->stream>>>(h->part, h->nblocks, c * kChunk, c == 0,
                                                   c == nchunks - 1, h->history, h->k1buf, h->k2buf,
                                                   h->dots, h->plan);
  }
  broyden_update_kernel<<<h->nblocks, kThreads, 0, h->stream>>>(
      x_in_dev, x_out_dev, h->f_old, h->x_old, h->V, h->W, h->len, h->history, h->zeta, h->plan,
      h->k1buf, h->k2buf, h->dots);
  broyden_advance_kernel<<<1, 1, 0, h->stream>>>(h->plan, h->history);
  NEGF_CUDA_TRY(cudaGetLastError());
  if (eps_max_host) {
    NEGF_CUDA_TRY(cudaMemcpyAsync(h->eps_pinned, &h->dots->eps_max, sizeof(double),
                                  cudaMemcpyDeviceToHost, h->stream));
    NEGF_CUDA_TRY(cudaStreamSynchronize(h->stream));
    *eps_max_host = *h->eps_pinned;
  }
  return NEGF_OK;
}
