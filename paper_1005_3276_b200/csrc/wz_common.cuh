// wz_common.cuh -- shared device-side types of the wz kernels: operator
// parameters, the device-resident CG state, and the fixed-order block/grid
// reduction with a "last block finalises" step (no host round trip, results
// independent of block scheduling order).
#pragma once
#include <cuda_runtime.h>

#include "wz_regfft.cuh"

namespace wz {

// Yukawa/mass and overlap parameters of Eq. (2.19).
template <typename R>
struct OpParams {
  R m_re, m_im;    // m
  R g2_re, g2_im;  // 2 g
  R rho;           // overlap parameter (paper: 1)
  int dagger;      // 0: M, 1: M^dag
  R shift;         // sigma: pass E' subtracts alpha (q + sigma p) (wz_cg_solve_shift)
  int pc;          // 1: site-local steps of the preconditioned operator Mtilde = 1 + Y M0^-1 (wz_p01.cuh)
};

// Device-resident scalars of one CG solve.
struct CGState {
  double bnorm2, bnorm;  // ||b||^2, ||b||
  double rr;             // rho_{k-1} = <r,r>
  double rr_new;         // rho_k candidate
  double pq;             // <p, M^dag M p> = ||M p||^2
  double alpha, beta;
  double rmax;           // max ||r|| since the last reliable update (G9)
  double tol, delta;
  double true_rr;        // ||b - A x||^2 recomputed
  double shift;          // sigma of the shifted system (M^dag M + sigma) x = b (0: plain)
  double pp;             // <p,p> of the current search direction (shifted solves)
  double aux;            // scratch norm (||b||^2 of the original system in preconditioned solves)
  int iter, max_iter;
  int n_ru;
  int converged;  // stop rule met
  int need_ru;    // reliable update requested; iteration kernels idle until served
  int stop;       // max_iter reached
  int use_ru;     // 1: complex64 vectors + reliable updates; 0: plain CG
  int pad_;
};

__device__ __forceinline__ bool cg_active(const CGState* st) {
  return !(st->converged | st->need_ru | st->stop);
}

// What the last block of a reduction does with the total.
enum { FIN_STORE = 0, FIN_PQ = 1, FIN_RR = 2, FIN_RU = 3, FIN_INIT = 4, FIN_TRUE = 5, FIN_AUX = 6, FIN_PP = 7, FIN_RRS = 8, FIN_HRU = 9 };
// FIN_HRU: reliable update of the binary16-storage solver (wz_cg_solve_half): the vectors were rescaled by f, st->aux = f^2
// and st->pp = the new scaled ||b|| were left by k_h_patch.
// FIN_PP / FIN_RRS select the shifted-system variants of passes A' / E' (wz_cg_solve_shift); FIN_RRS
// finalises like FIN_RR.

template <int FIN>
__device__ __forceinline__ void cg_finalize(double total, CGState* st, double* store) {
  if (FIN == FIN_STORE) {
    *store = total;
  } else if (FIN == FIN_PQ) {  // alpha = rho_{k-1} / <p, A p>
    st->pq = total + st->shift * st->pp;  // <p, (A + sigma) p> = ||M p||^2 + sigma <p,p>
    st->alpha = st->rr / st->pq;
  } else if (FIN == FIN_INIT) {  // r0 = p0 = b
    st->bnorm2 = total;
    st->bnorm = sqrt(total);
    st->rr = total;
    st->rmax = sqrt(total);
    if (total == 0.0) st->converged = 1;
  } else if (FIN == FIN_RR || FIN == FIN_RRS) {  // after x += alpha p, r -= alpha q
    const double rn = sqrt(total);
    st->iter += 1;
    if (st->use_ru) {
      if (rn > st->rmax) st->rmax = rn;
      if (rn < st->delta * st->rmax || rn <= st->tol * st->bnorm) {
        st->rr_new = total;
        st->need_ru = 1;
      } else {
        st->beta = total / st->rr;
        st->rr = total;
      }
    } else {
      if (rn <= st->tol * st->bnorm) {
        st->converged = 1;
      } else {
        st->beta = total / st->rr;
      }
      st->rr = total;
    }
    if (!st->converged && !st->need_ru && st->iter >= st->max_iter) st->stop = 1;
  } else if (FIN == FIN_RU) {  // r = b - A X recomputed in complex128
    const double rn = sqrt(total);
    st->n_ru += 1;
    st->rmax = rn;
    st->true_rr = total;
    if (rn <= st->tol * st->bnorm) st->converged = 1;
    st->beta = total / st->rr;
    st->rr = total;
    st->need_ru = 0;
    if (!st->converged && st->iter >= st->max_iter) st->stop = 1;
  } else if (FIN == FIN_HRU) {  // r = s' (b - A X) as stored in binary16, p rescaled by f = s'/s
    st->n_ru += 1;
    st->rmax = sqrt(total);
    st->true_rr = total;
    st->beta = total / (st->aux * st->rr);  // rho_{k-1} in the new units
    st->rr = total;
    st->bnorm = st->pp;
    st->need_ru = 0;
    if (st->iter >= st->max_iter) st->stop = 1;
  } else if (FIN == FIN_TRUE) {
    st->true_rr = total;
  } else if (FIN == FIN_AUX) {
    st->aux = total;
  } else if (FIN == FIN_PP) {
    st->pp = total;
  }
}

// Reduction workspace: one partial per block, a ticket counter, and the target.
// Batched solves keep one CGState, one counter and one row of partials PER SOURCE; a
// kernel working on source `src` uses for_source(src).
struct RedArgs {
  double* partials;   // [nsources][pstride]
  unsigned* counter;  // [nsources]; zero before first use; left zero after each use
  CGState* st;        // [nsources]
  double* store;      // FIN_STORE target, [nsources]
  int pstride;
  __host__ __device__ RedArgs for_source(int src) const {
    RedArgs r = *this;
    r.partials = partials ? partials + (long)src * pstride : nullptr;
    r.counter = counter ? counter + src : nullptr;
    r.st = st ? st + src : nullptr;
    r.store = store ? store + src : nullptr;
    return r;
  }
};

// Sum `v` over the block in a fixed order; returns the total in thread 0.
__device__ __forceinline__ double block_sum(double v, double* sh /* >= 32 doubles */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (lane == 0) sh[wid] = v;
  __syncthreads();
  double t = 0.0;
  if (wid == 0) {
    t = (lane < nw) ? sh[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
  }
  return t;
}

// Each block contributes `v` (per thread); the last block to arrive sums all
// partials in index order and runs cg_finalize<FIN>.  `blk`/`nblk`: linear block id
// and count.  All threads of the block must call this.
template <int FIN>
__device__ __forceinline__ void grid_reduce(double v, const RedArgs& ra, int blk, int nblk,
                                            double* sh /* >= 33 doubles */) {
  double t = block_sum(v, sh);
  __shared__ int s_last;
  if (threadIdx.x == 0) {
    ra.partials[blk] = t;
    __threadfence();
    unsigned ticket = atomicAdd(ra.counter, 1u);
    s_last = (ticket == (unsigned)(nblk - 1));
  }
  __syncthreads();
  if (s_last) {
    __threadfence();
    double acc = 0.0;
    for (int i = threadIdx.x; i < nblk; i += blockDim.x) acc += __ldcg(ra.partials + i);
    double tot = block_sum(acc, sh);
    if (threadIdx.x == 0) {
      cg_finalize<FIN>(tot, ra.st, ra.store);
      *ra.counter = 0u;
      __threadfence();
    }
  }
}

// The pass kernels (wz_p01.cuh) only leave their per-CTA partial: with one 512-thread CTA per SM, waiting for the
// ticket (fence + atomic round trip) kept the whole SM idle for ~1 us per CTA, 6-7 % of passes C and E' (ncu source
// view, profiles/r02_*).  The total and the scalar update are taken by k_finalize, a one-CTA-per-source launch
// right behind the pass (wz_lib.cu: launch_p01); same fixed order of summation, no atomics.
__device__ __forceinline__ void block_partial(double v, const RedArgs& ra, int blk, double* sh) {
  double t = block_sum(v, sh);
  if (threadIdx.x == 0) ra.partials[blk] = t;
}

constexpr int FINALIZE_NT = 256;
template <int FIN>
__global__ void __launch_bounds__(FINALIZE_NT) k_finalize(RedArgs red, int nblk, const CGState* gate) {
  const int src = blockIdx.x;
  if (gate && !cg_active(gate + src)) return;  // an idle source: its CTAs returned before writing partials
  const RedArgs ra = red.for_source(src);
  __shared__ double sh[33];
  double acc = 0.0;
  for (int i = threadIdx.x; i < nblk; i += blockDim.x) acc += ra.partials[i];
  const double tot = block_sum(acc, sh);
  if (threadIdx.x == 0) cg_finalize<FIN>(tot, ra.st, ra.store);
}

}  // namespace wz
