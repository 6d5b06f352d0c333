// wz_p01p.cuh -- persistent, software-pipelined version of the strided (x0, x1) pass
// (wz_p01.cuh explains the modes).  One CTA per SM loops over tiles; the operand
// tiles of the NEXT tile are fetched with cp.async (LDGSTS, 16-byte chunks, no
// registers) into the other half of a two-stage shared-memory ring while the
// current tile is transformed, so HBM latency overlaps the butterflies instead of
// adding to them (profiles/r01_*: the non-pipelined pass is the sum of its phases).
//
// Stage layout (elements): S0 = main tile, padded [x0][PITCH0] (also the exchange
// buffer between the two axes), S1/S2 = site-local operand tiles, dense [x0][x1][s].
#pragma once
#include "wz_p01.cuh"

namespace wz {

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <typename R, int L0, int L1, int NSEG, int T0, int T1, int MODE>
struct P01PCfg {
  using Base = P01Cfg<R, L0, L1, NSEG, T0, T1>;
  static constexpr int NT = Base::NT;
  static constexpr int PITCH0 = Base::PITCH0;
  static constexpr int NS1 = (MODE == P01_MID || MODE == P01_END || MODE == P01_ENDCG || MODE == P01_FWDCG) ? 2 : 0;
  static constexpr int S0_ELEMS = L0 * PITCH0;
  static constexpr int S1_ELEMS = L0 * L1 * NSEG;
  static constexpr int STAGE_ELEMS = S0_ELEMS + NS1 * S1_ELEMS;
  static constexpr size_t SMEM = sizeof(cpx<R>) * 2 * (size_t)STAGE_ELEMS;
  static constexpr int CPR = NSEG * (int)sizeof(cpx<R>) / 16;  // 16-byte chunks per (x0,x1) row
  static_assert(NSEG * sizeof(cpx<R>) % 16 == 0, "rows must be multiples of 16 bytes");
};

// copy one L0 x L1 x NSEG tile (rows of NSEG elements, row stride I in global memory)
template <typename R, int L0, int L1, int NSEG, int NT, int DST_PITCH0>
__device__ __forceinline__ void tile_prefetch(cpx<R>* sdst, const cpx<R>* gsrc, long I, int tid) {
  constexpr int CPR = NSEG * (int)sizeof(cpx<R>) / 16;
  constexpr int EPC = 16 / (int)sizeof(cpx<R>);  // elements per chunk
  constexpr int NCH = L0 * L1 * CPR;
#pragma unroll
  for (int c0 = 0; c0 < NCH; c0 += NT) {
    const int c = c0 + tid;
    if (NCH % NT == 0 || c < NCH) {
      const int row = c / CPR, part = c % CPR;
      const int x0 = row / L1, x1 = row % L1;
      cp_async16(sdst + x0 * DST_PITCH0 + x1 * NSEG + part * EPC, gsrc + (long)row * I + part * EPC);
    }
  }
}

template <typename R, int L0, int L1, int NSEG, int T0, int T1, int MODE, int FIN>
__global__ void __launch_bounds__(P01PCfg<R, L0, L1, NSEG, T0, T1, MODE>::NT, 1)
k_p01p(const P01Args<R> a, const int nseg_tiles, const int ntiles) {
  using Cfg = P01PCfg<R, L0, L1, NSEG, T0, T1, MODE>;
  constexpr int NT = Cfg::NT, PITCH0 = Cfg::PITCH0;
  constexpr int NR0 = L0 / T0, NR1 = L1 / T1;
  constexpr int TWSTEP = TWN / 2 / L0;
  constexpr bool kFwd = (MODE == P01_FWD || MODE == P01_FWDCG);
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cpx<R>* sm = reinterpret_cast<cpx<R>*>(smem_raw);
  __shared__ double red_sh[33];

  if (a.gate && !cg_active(a.gate)) return;

  const int tid = threadIdx.x;
  const long V = (long)L0 * L1 * a.I;
  int lineA, jA, lineB, jB;
  lane_split<T0>(tid, lineA, jA);
  lane_split<T1>(tid, lineB, jB);
  const bool actA = lineA < L1 * NSEG;
  const int x1A = lineA / NSEG, sA = lineA % NSEG;
  const bool actB = lineB < L0 * NSEG;
  const int x0B = lineB / NSEG, sB = lineB % NSEG;

  // tile t -> (segment, field): neighbouring CTAs work on neighbouring segments
  auto issue = [&](int t, int stage) {
    const int seg = t % nseg_tiles, f = t / nseg_tiles;
    const long base = (long)f * V + (long)seg * NSEG;
    cpx<R>* st = sm + stage * Cfg::STAGE_ELEMS;
    const cpx<R>* main_src = (MODE == P01_FWDCG) ? a.cg_p : a.in;
    tile_prefetch<R, L0, L1, NSEG, NT, PITCH0>(st, main_src + base, a.I, tid);
    if constexpr (MODE == P01_FWDCG) {
      tile_prefetch<R, L0, L1, NSEG, NT, L1 * NSEG>(st + Cfg::S0_ELEMS, a.cg_r + base, a.I, tid);
      tile_prefetch<R, L0, L1, NSEG, NT, L1 * NSEG>(st + Cfg::S0_ELEMS + Cfg::S1_ELEMS, a.cg_x + base, a.I, tid);
    } else if constexpr (Cfg::NS1 == 2) {
      tile_prefetch<R, L0, L1, NSEG, NT, L1 * NSEG>(st + Cfg::S0_ELEMS, a.psi + base, a.I, tid);
      tile_prefetch<R, L0, L1, NSEG, NT, L1 * NSEG>(st + Cfg::S0_ELEMS + Cfg::S1_ELEMS,
                                                    a.phi + (long)seg * NSEG, a.I, tid);
    }
  };

  double acc = 0.0;
  int t = blockIdx.x, stage = 0;
  if (t < ntiles) issue(t, 0);
  cp_async_commit();
  for (; t < ntiles; t += gridDim.x, stage ^= 1) {
    const int tn = t + gridDim.x;
    if (tn < ntiles) issue(tn, stage ^ 1);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();

    const int seg = t % nseg_tiles, f = t / nseg_tiles;
    const int comp = f & 3;
    const long base = (long)f * V + (long)seg * NSEG;
    cpx<R>* s0 = sm + stage * Cfg::STAGE_ELEMS;
    const cpx<R>* s1 = s0 + Cfg::S0_ELEMS;
    const cpx<R>* s2 = s1 + Cfg::S1_ELEMS;
    cpx<R>* gout = a.out + base;

    if constexpr (kFwd) {
      using F0 = LineFFT<R, L0, +1, VAR_DIT, T0>;
      using F1 = LineFFT<R, L1, +1, VAR_DIT, T1>;
      cpx<R> x[NR0];
      R alpha = R(0), beta = R(0);
      if constexpr (MODE == P01_FWDCG) {
        alpha = (R)a.gate->alpha;
        beta = (R)a.gate->beta;
      }
#pragma unroll
      for (int k = 0; k < NR0; ++k) {
        const int x0 = F0::in_pos(k, jA);
        cpx<R> v = {R(0), R(0)};
        if (actA) {
          v = s0[x0 * PITCH0 + x1A * NSEG + sA];
          if constexpr (MODE == P01_FWDCG) {
            // x += alpha p (pending update of the previous iteration); p <- r + beta p
            const int d = (x0 * L1 + x1A) * NSEG + sA;
            const long off = base + ((long)x0 * L1 + x1A) * a.I + sA;
            const cpx<R> vr = s1[d], vx = s2[d];
            a.cg_x[off] = {vx.re + alpha * v.re, vx.im + alpha * v.im};
            v = {vr.re + beta * v.re, vr.im + beta * v.im};
            a.cg_p[off] = v;
          }
        }
        if (a.apbc) v = mul_tw_rt<R, +1>(v, x0 * TWSTEP);
        x[k] = v;
      }
      F0::run(x, jA);
      __syncthreads();  // every read of the landed tile is done
      if (actA) {
#pragma unroll
        for (int k = 0; k < NR0; ++k) s0[F0::out_pos(k, jA) * PITCH0 + x1A * NSEG + sA] = x[k];
      }
      __syncthreads();
      cpx<R> y[NR1];
#pragma unroll
      for (int k = 0; k < NR1; ++k) {
        cpx<R> v = {R(0), R(0)};
        if (actB) v = s0[x0B * PITCH0 + F1::in_pos(k, jB) * NSEG + sB];
        y[k] = v;
      }
      F1::run(y, jB);
      if (actB) {
#pragma unroll
        for (int k = 0; k < NR1; ++k) gout[((long)x0B * L1 + F1::out_pos(k, jB)) * a.I + sB] = y[k];
      }
    } else {
      using G1 = LineFFT<R, L1, -1, VAR_DIT, T1>;
      using G0 = LineFFT<R, L0, -1, VAR_DIT, T0>;
      {
        cpx<R> y[NR1];
#pragma unroll
        for (int k = 0; k < NR1; ++k) {
          cpx<R> v = {R(0), R(0)};
          if (actB) v = s0[x0B * PITCH0 + G1::in_pos(k, jB) * NSEG + sB];
          y[k] = v;
        }
        G1::run(y, jB);
        __syncthreads();
        if (actB) {
#pragma unroll
          for (int k = 0; k < NR1; ++k) s0[x0B * PITCH0 + G1::out_pos(k, jB) * NSEG + sB] = y[k];
        }
      }
      __syncthreads();
      cpx<R> x[NR0];
      cpx<R> vr[(MODE == P01_ENDCG) ? NR0 : 1];
#pragma unroll
      for (int k = 0; k < NR0; ++k) {
        cpx<R> v = {R(0), R(0)};
        if (actA) v = s0[G0::in_pos(k, jA) * PITCH0 + x1A * NSEG + sA];
        x[k] = v;
      }
      if constexpr (MODE == P01_ENDCG) {
        // r of this thread's sites: in flight while the axis-0 butterflies run
#pragma unroll
        for (int k = 0; k < NR0; ++k) {
          cpx<R> v = {R(0), R(0)};
          if (actA) v = a.cg_r[base + ((long)G0::out_pos(k, jA) * L1 + x1A) * a.I + sA];
          vr[k] = v;
        }
      }
      G0::run(x, jA);
#pragma unroll
      for (int k = 0; k < NR0; ++k) {
        const int x0 = G0::out_pos(k, jA);
        cpx<R> v = x[k];
        if (a.apbc) v = mul_tw_rt<R, -1>(v, x0 * TWSTEP);
        x[k] = cscale(v, a.scale);
      }
      if constexpr (MODE == P01_INV) {
        if (actA) {
#pragma unroll
          for (int k = 0; k < NR0; ++k) gout[((long)G0::out_pos(k, jA) * L1 + x1A) * a.I + sA] = x[k];
        }
      } else {
        // site-local term of Eq. (2.19), operands from the staged dense tiles
        const bool use_conj = (comp < 2) != (a.op.dagger != 0);
        R alpha = R(0);
        if constexpr (MODE == P01_ENDCG) alpha = (R)a.red.st->alpha;
        if (actA) {
#pragma unroll
          for (int k = 0; k < NR0; ++k) {
            const int x0 = G0::out_pos(k, jA);
            const int d = (x0 * L1 + x1A) * NSEG + sA;
            const long off = base + ((long)x0 * L1 + x1A) * a.I + sA;
            const cpx<R> ps = s1[d], ph = s2[d];
            cpx<R> w = {a.op.m_re + a.op.g2_re * ph.re - a.op.g2_im * ph.im,
                        a.op.m_im + a.op.g2_re * ph.im + a.op.g2_im * ph.re};
            if (use_conj) w.im = -w.im;
            cpx<R> v = x[k];
            v.re += w.re * ps.re - w.im * ps.im;
            v.im += w.re * ps.im + w.im * ps.re;
            if constexpr (MODE == P01_ENDCG) {
              const cpx<R> rn = {vr[k].re - alpha * v.re, vr[k].im - alpha * v.im};
              a.cg_r[off] = rn;
              acc += (double)rn.re * (double)rn.re + (double)rn.im * (double)rn.im;
            } else {
              x[k] = v;
              a.site_out[off] = v;
              if (FIN != FIN_STORE || a.red.partials)
                acc += (double)v.re * (double)v.re + (double)v.im * (double)v.im;
            }
          }
        }
        if constexpr (MODE == P01_MID) {
          using F0 = LineFFT<R, L0, +1, VAR_DIF, T0>;
          using F1 = LineFFT<R, L1, +1, VAR_DIT, T1>;
          cpx<R> z[NR0];
#pragma unroll
          for (int k = 0; k < NR0; ++k) {
            const int x0 = G0::out_pos(k, jA);
            cpx<R> v = x[k];
            if (a.apbc) v = mul_tw_rt<R, +1>(v, x0 * TWSTEP);
            z[out_index<NR0>(k)] = v;
          }
          F0::run(z, jA);
          __syncthreads();
          if (actA) {
#pragma unroll
            for (int k = 0; k < NR0; ++k) s0[F0::out_pos(k, jA) * PITCH0 + x1A * NSEG + sA] = z[k];
          }
          __syncthreads();
          cpx<R> y[NR1];
#pragma unroll
          for (int k = 0; k < NR1; ++k) {
            cpx<R> v = {R(0), R(0)};
            if (actB) v = s0[x0B * PITCH0 + F1::in_pos(k, jB) * NSEG + sB];
            y[k] = v;
          }
          F1::run(y, jB);
          if (actB) {
#pragma unroll
            for (int k = 0; k < NR1; ++k) gout[((long)x0B * L1 + F1::out_pos(k, jB)) * a.I + sB] = y[k];
          }
        }
      }
    }
    __syncthreads();  // this stage may be refilled by the next iteration's prefetch
  }
  cp_async_wait<0>();
  if constexpr (MODE == P01_MID || MODE == P01_END || MODE == P01_ENDCG) {
    if (a.red.partials) grid_reduce<FIN>(acc, a.red, blockIdx.x, gridDim.x, red_sh);
  }
}

}  // namespace wz
