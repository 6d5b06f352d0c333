// wz_p01.cuh -- the strided two-axis pass: DFTs over axes (x0, x1) of one spin
// component, for a tile of NSEG consecutive values of the flattened (x2,x3) index.
//
// Modes (SURVEY 7.2 passes A, C, E; steps a1, a2, a4, a5, a6 of SURVEY 8(a)):
//   P01_FWD : [time pre-twist] -> DFT axis 0 -> DFT axis 1                   (pass A)
//   P01_INV : inverse DFT axis 1 -> inverse DFT axis 0 -> [post-twist] * scale
//   P01_MID : P01_INV, then  chi = t + W psi  (Yukawa + mass, Eq. 2.19), store chi,
//             [accumulate ||chi||^2], then P01_FWD on chi                    (pass C)
//   P01_END : P01_INV, then  out = t + W psi, store out                      (pass E)
// Each thread (or lane pair) owns one lattice line in registers; the only shared
// memory traffic is one write + one read per element per axis change.
#pragma once
#include "wz_common.cuh"

namespace wz {

enum { P01_FWD = 0, P01_INV = 1, P01_MID = 2, P01_END = 3, P01_FWDCG = 4, P01_ENDCG = 5 };
// CG-fused variants (SURVEY 7.2 "CG fusion"; steps a8-a10 of SURVEY 8(a)):
//   P01_FWDCG : on load  x += alpha p (the update left pending by the previous iteration),
//               p <- r + beta p (both stored back), then P01_FWD on p
//   P01_ENDCG : P01_INV, q = t + W chi (never stored);  r -= alpha q;
//               ||r||^2 -> FIN_RR (stop rule, beta, reliable-update request)
// x lags by one update: wz_lib.cu flushes it (k_flush_x) before x is used.

__device__ __forceinline__ cpx<float> ldg_c(const cpx<float>* p) {
  float2 t = __ldg(reinterpret_cast<const float2*>(p));
  return {t.x, t.y};
}
__device__ __forceinline__ cpx<double> ldg_c(const cpx<double>* p) {
  double2 t = __ldg(reinterpret_cast<const double2*>(p));
  return {t.x, t.y};
}

// Streaming loads: chi in passes E / E' is read once and by no launch soon after; marking it evict-first
// in L2 (createpolicy + .L2::cache_hint) leaves more of the 126 MB L2 to what the NEXT launch reads first
// (the tail of r written here; see next_sweep() in wz_lib.cu).  Measured at 32^4 complex64, 12 sources:
// pass E' 307.6 -> 291 us per launch.  The same hint on x / r in pass A' and on the chi store of pass C
// made those passes slower (420 -> 599 us, 380 -> 406 us; round-1 A/B runs) and is not used.
#ifndef WZ_EVICT
#define WZ_EVICT 1
#endif
#ifndef WZ_EVICT_MID
#define WZ_EVICT_MID 0
#endif
__device__ __forceinline__ unsigned long long l2_evict_first_policy() {
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ cpx<float> ld_stream(const cpx<float>* p, unsigned long long pol) {
#if WZ_EVICT
  cpx<float> v;
  asm volatile("ld.global.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.re), "=f"(v.im) : "l"(p), "l"(pol));
  return v;
#else
  return *p;
#endif
}
__device__ __forceinline__ cpx<double> ld_stream(const cpx<double>* p, unsigned long long pol) {
#if WZ_EVICT
  cpx<double> v;
  asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.re), "=d"(v.im) : "l"(p), "l"(pol));
  return v;
#else
  return *p;
#endif
}
// read-only data (non-coherent path, as ldg_c)
__device__ __forceinline__ cpx<float> ld_stream_nc(const cpx<float>* p, unsigned long long pol) {
#if WZ_EVICT
  cpx<float> v;
  asm volatile("ld.global.nc.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.re), "=f"(v.im) : "l"(p), "l"(pol));
  return v;
#else
  return ldg_c(p);
#endif
}
__device__ __forceinline__ cpx<double> ld_stream_nc(const cpx<double>* p, unsigned long long pol) {
#if WZ_EVICT
  cpx<double> v;
  asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.re), "=d"(v.im) : "l"(p), "l"(pol));
  return v;
#else
  return ldg_c(p);
#endif
}
__device__ __forceinline__ void st_stream(cpx<float>* p, cpx<float> v, unsigned long long pol) {
#if WZ_EVICT
  asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.re), "f"(v.im), "l"(pol));
#else
  *p = v;
#endif
}
__device__ __forceinline__ void st_stream(cpx<double>* p, cpx<double> v, unsigned long long pol) {
#if WZ_EVICT
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.re), "d"(v.im), "l"(pol));
#else
  *p = v;
#endif
}

// L2 prefetch hint: no register, no scoreboard; the later load then pays L2 latency
// instead of HBM latency (the passes are latency-bound on their operand streams).
__device__ __forceinline__ void prefetch_l2(const void* p) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
// narrower storage (SProxy, wz_regfft.cuh): same helpers, converting
template <typename R, typename S>
__device__ __forceinline__ void prefetch_l2(SProxy<R, S> p) { prefetch_l2(p.raw()); }
template <typename R, typename S>
__device__ __forceinline__ cpx<R> ldg_c(SProxy<R, S> p) {
  const unsigned u = __ldg(reinterpret_cast<const unsigned*>(p.raw()));
  const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&u));
  return {(R)f.x, (R)f.y};
}
template <typename R, typename S>
__device__ __forceinline__ cpx<R> ld_stream_nc(SProxy<R, S> p, unsigned long long pol) {
  unsigned u;
  asm volatile("ld.global.nc.L2::cache_hint.b32 %0, [%1], %2;" : "=r"(u) : "l"(p.raw()), "l"(pol));
  const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&u));
  return {(R)f.x, (R)f.y};
}

// A CUtensorMap (TMA descriptor) carried by value in the kernel parameters; encoded on the host
// (wz_lib.cu: make_tile_tmap).  Used only to PREFETCH whole strided tiles into L2, one instruction per tile.
struct alignas(64) TMapBlob {
  unsigned long long v[16];
};
// L2 prefetch of the box at (c0, c1, c2, c3) of a rank-4 tiled tensor map (innermost coordinate first).
__device__ __forceinline__ void tma_prefetch_l2_4d(const TMapBlob* tm, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];"
               ::"l"(reinterpret_cast<unsigned long long>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
               : "memory");
}

template <typename R>
struct P01Args {
  const cpx<R>* in;   // [nf][L0][L1][I]
  cpx<R>* out;        // same shape (may alias in)
  long I;             // L2*L3
  int apbc;           // antiperiodic time twist on/off
  R scale;            // 1/V for the inverse modes; binary16 storage: 1/(L0 L1), applied before the forward transforms
  // MID / END only:
  const cpx<R>* psi;  // operand of the site-local term (psi for MID, chi for END)
  const cpx<R>* phi;  // [L0][L1][I]
  cpx<R>* site_out;   // chi (MID) or the matvec result (END)
  OpParams<R> op;
  RedArgs red;        // MID: ||chi||^2 (partials == nullptr: skip);  ENDCG: ||r||^2
  cpx<R>* cg_r;       // FWDCG (read), ENDCG (read+write)
  cpx<R>* cg_p;       // FWDCG (read+write), ENDCG (read)
  cpx<R>* cg_x;       // FWDCG (read+write)
  const CGState* gate;  // [nbatch]; if set and this source's solve is idle, the CTA returns at once
  int rev;              // 1: CTAs take the tiles in reverse order (see launch_p01: L2 reuse across launches)
  int fdiv;             // fields per (source, spin) pair: 1, or L0 when the x0 slices are passed as separate fields
                        //    (the axis-1 sub-pass of the single-axis decomposition); 0 is read as 1
  // Wave-ahead tile prefetch (passes C, A'): tm_in describes `in` as [nf][L0][L1][2*I reals] with a box of one
  // tile; the CTA prefetches the input tile of the CTA tm_ahead launches further on (one wave of resident CTAs)
  // into L2 with ONE TMA instruction, so that CTA later pays L2 instead of HBM latency for its first loads.
  TMapBlob tm_in;
  int tm_ahead;         // 0: off
  int comp_fast;        // 1: launch order = (source, tile, spin) with spin fastest: the four CTAs that share one
                        //    phi tile run together, so phi comes from HBM once per source instead of four times
};

template <typename R, int L0, int L1, int NSEG, int T0, int T1>
struct P01Cfg {
  static constexpr int TPL0 = T0, TPL1 = T1;  // lanes per line along axis 0 / axis 1
  static constexpr int NR0 = L0 / TPL0, NR1 = L1 / TPL1;
  static constexpr int NT_A = L1 * NSEG * TPL0;  // threads when lines run along axis 0
  static constexpr int NT_B = L0 * NSEG * TPL1;  // threads when lines run along axis 1
  // L1 == 1: a single-axis pass (lines along axis 0 only, no tile exchange): the decomposition of the 64x64
  // lattices, where a two-axis tile with runs longer than 32 bytes does not fit (wz_lib.cu: split01)
  static constexpr int NT_RAW = (L1 == 1) ? NT_A : (NT_A > NT_B ? NT_A : NT_B);
  static constexpr int NT = (NT_RAW + 31) / 32 * 32;
  static constexpr int PITCH0 = L1 * NSEG + NSEG;  // padded x0 stride (elements)
  static constexpr size_t SMEM = (L1 == 1) ? 0 : sizeof(cpx<R>) * (size_t)L0 * PITCH0;
};

// Resident CTAs per SM the register allocation must allow: 32x32 complex64 tiles aim at
// 1024 resident threads per SM (64 registers each); everything else takes what it needs.
template <typename R, int L0, int L1, int NT, int TPL>
struct p01_minb {  // TPL = 2: 16 values per thread, 64 registers; TPL = 1: 32 values, 128 registers
  static constexpr int want = 512 * TPL;
  static constexpr int v = (sizeof(R) == 4 && L0 == 32 && L1 == 32 && NT <= want) ? (want / NT) : 1;
};

// Where the total of a reduction is taken.  Large tiles (one or two big CTAs per SM, hundreds of microseconds per
// launch): the pass leaves per-CTA partials and a one-CTA-per-source kernel right behind it takes the total (the
// fence + ticket round trip of the in-kernel version kept the SM idle ~1 us per CTA: 6-7 % of passes C and E' at
// 32^4).  Small tiles (launch-bound lattices, a few microseconds per launch): the last CTA to arrive takes the total
// inside the pass (one kernel node fewer per reduction in the iteration graph).
template <int L0, int L1>
struct p01_split_finalize {
  static constexpr bool v = (L0 * L1 >= 1024) || L1 == 1;
};

template <typename R, int L0, int L1, int NSEG, int T0, int T1, int MODE, int FIN, int IC = 0, typename S = cpx<R>>
__global__ void __launch_bounds__(P01Cfg<R, L0, L1, NSEG, T0, T1>::NT, p01_minb<R, L0, L1, P01Cfg<R, L0, L1, NSEG, T0, T1>::NT, T0>::v)
k_p01(const __grid_constant__ P01Args<R> a) {
  using Cfg = P01Cfg<R, L0, L1, NSEG, T0, T1>;
  constexpr int TPL0 = Cfg::TPL0, TPL1 = Cfg::TPL1, NR0 = Cfg::NR0, NR1 = Cfg::NR1;
  constexpr int PITCH0 = Cfg::PITCH0;
  constexpr int TWSTEP = TWN / 2 / L0;  // twist exp(-i pi x0/L0) = table[x0 * TWSTEP]
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cpx<R>* sm = reinterpret_cast<cpx<R>*>(smem_raw);
  __shared__ double red_sh[33];

  const int tid = threadIdx.x;
  [[maybe_unused]] const unsigned long long pol = l2_evict_first_policy();
  // sweep direction: with rev the first CTAs of this launch take what the previous launch wrote last
  int bx = a.rev ? (int)(gridDim.x - 1 - blockIdx.x) : (int)blockIdx.x;
  int f = a.rev ? (int)(gridDim.y - 1 - blockIdx.y) : (int)blockIdx.y;  // field = source*4 + spin
  if (a.comp_fast) {
    const unsigned lin0 = blockIdx.y * gridDim.x + blockIdx.x;
    const unsigned lin = a.rev ? gridDim.x * gridDim.y - 1 - lin0 : lin0;
    const unsigned q = lin >> 2;
    bx = (int)(q % gridDim.x);
    f = (int)(q / gridDim.x) * 4 + (int)(lin & 3);
  }
  const int fq = (a.fdiv > 1) ? f / a.fdiv : f;
  const int comp = fq & 3, src = fq >> 2;
  // forward modes: the idle test of this source is issued now but consumed only after the
  // first loads are in flight (measured: pays there, not in the inverse modes)
  int idle = 0;
  if (a.gate) idle = a.gate[src].converged | a.gate[src].need_ru | a.gate[src].stop;
  if constexpr (MODE != P01_FWD && MODE != P01_FWDCG) {
    if (idle) return;
  }
  const long i0 = (long)bx * NSEG;
  // IC > 0: the (x2,x3) volume is a compile-time constant, so every tile offset below folds
  // into an immediate of the load/store instead of 64-bit integer arithmetic per access
  const long I = IC ? (long)IC : a.I;
  const long V = (long)L0 * L1 * I;
  // S: how t, chi, r, p are STORED (cpx<R>, or cpxh = two binary16 values); x and phi are always cpx<R>
  using VP = typename sptr<R, S>::type;
  const VP gin = as_stored<R, S>(a.in) + ((long)f * V + i0);
  const VP gout = as_stored<R, S>(a.out) + ((long)f * V + i0);
  [[maybe_unused]] const VP s_r = as_stored<R, S>(a.cg_r);
  [[maybe_unused]] const VP s_p = as_stored<R, S>(a.cg_p);

  // thread roles: A = line along axis 0 at (x1, s); B = line along axis 1 at (x0, s)
  int lineA, jA, lineB, jB;
  lane_split<TPL0>(tid, lineA, jA);
  lane_split<TPL1>(tid, lineB, jB);
  const bool actA = lineA < L1 * NSEG;
  const int x1A = lineA / NSEG, sA = lineA % NSEG;
  const bool actB = lineB < L0 * NSEG;
  const int x0B = lineB / NSEG, sB = lineB % NSEG;

  // Passes C and A', issued LATE in the CTA's life (C: before its forward half, about a quarter of its time left;
  // A': the tile of p, before the transforms): the CTA
  // tm_ahead launches further on takes over an SM a few microseconds later.  Measured at 32^4 x 12: pass C 360 -> 339 us.
  // (Issued at the start, a whole wave early, the tiles were evicted again by the ~80 MB that stream through L2 per
  // wave and came from HBM twice: 360 -> 396 us.  Pass E' gains nothing at any issue point, 306 -> 306...329 us; pass A'
  // 445 -> 436 us.  Prefetching the operand tiles (r, x; p, phi) the same way lost: C 342 -> 366, A' 436 -> 467 us.)
  auto prefetch_next_tile = [&]() {
    if (a.tm_ahead > 0 && tid == 0) {
      const unsigned tot = gridDim.x * gridDim.y;
      const unsigned l2 = blockIdx.y * gridDim.x + blockIdx.x + (unsigned)a.tm_ahead;  // launch order, x fastest
      if (l2 < tot) {
        int bx2, f2;  // the same launch-order -> (tile, field) map as above
        if (a.comp_fast) {
          const unsigned lin = a.rev ? tot - 1 - l2 : l2;
          const unsigned q = lin >> 2;
          bx2 = (int)(q % gridDim.x);
          f2 = (int)(q / gridDim.x) * 4 + (int)(lin & 3);
        } else {
          const unsigned xr = l2 % gridDim.x, yr = l2 / gridDim.x;
          bx2 = a.rev ? (int)(gridDim.x - 1 - xr) : (int)xr;
          f2 = a.rev ? (int)(gridDim.y - 1 - yr) : (int)yr;
        }
        tma_prefetch_l2_4d(&a.tm_in, 2 * bx2 * NSEG, 0, 0, f2);
      }
    }
  };
  if constexpr (MODE == P01_FWD || MODE == P01_FWDCG) {
    using F0 = LineFFT<R, L0, +1, VAR_DIT, TPL0>;
    using F1 = LineFFT<R, L1, +1, VAR_DIT, TPL1>;
    cpx<R> x[NR0];
    [[maybe_unused]] double accp = 0.0;  // ||p||^2 of the new search direction (FIN_PP: shifted solves)
    if constexpr (MODE == P01_FWDCG) {
      // p <- r + beta p (PAPER.md:896 CG), all p loads first, r through the
      // read-only path so that nothing waits behind the p stores
      const long fo = (long)f * V + i0;
      if (actA && (sA * (int)sizeof(cpx<R>)) % 32 == 0) {
#pragma unroll
        for (int k = 0; k < NR0; ++k) {
          const long off = fo + ((long)F0::in_pos(k, jA) * L1 + x1A) * I + sA;
          prefetch_l2(s_r + off);
          prefetch_l2(a.cg_x + off);
        }
      }
#pragma unroll
      for (int k = 0; k < NR0; ++k) {
        cpx<R> v = {R(0), R(0)};
        if (actA) v = s_p[fo + ((long)F0::in_pos(k, jA) * L1 + x1A) * I + sA];
        x[k] = v;
      }
      const R beta = (R)a.gate[src].beta, alpha = (R)a.gate[src].alpha;
      if (idle) return;
      constexpr int CHF = (NR0 % 8 == 0) ? 8 : 4;
#pragma unroll
      for (int k0 = 0; k0 < NR0; k0 += CHF) {
        cpx<R> vr[CHF], vx[CHF];
        long off[CHF];
#pragma unroll
        for (int c = 0; c < CHF; ++c) {
          off[c] = fo + ((long)F0::in_pos(k0 + c, jA) * L1 + x1A) * I + sA;
          vr[c] = {R(0), R(0)};
          vx[c] = {R(0), R(0)};
          if (actA) {
            vr[c] = ldg_c(s_r + off[c]);
            vx[c] = a.cg_x[off[c]];  // read, then written, by this thread only
          }
        }
#pragma unroll
        for (int c = 0; c < CHF; ++c) {
          const int x0 = F0::in_pos(k0 + c, jA);
          cpx<R> v = x[k0 + c];
          if (actA) {
            a.cg_x[off[c]] = {vx[c].re + alpha * v.re, vx[c].im + alpha * v.im};  // pending x += alpha p
            v = as_if_stored<R, S>({vr[c].re + beta * v.re, vr[c].im + beta * v.im});  // narrower storage: transform what is stored
            s_p[off[c]] = v;
            if constexpr (FIN == FIN_PP) accp += (double)v.re * (double)v.re + (double)v.im * (double)v.im;
          }
          if constexpr (sizeof(S) != sizeof(cpx<R>)) v = cscale(v, a.scale);  // binary16 storage: 1/(L0 L1) here, 1/(L2 L3) in the multiply pass
          if (a.apbc) v = mul_tw_rt<R, +1>(v, x0 * TWSTEP);
          x[k0 + c] = v;
        }
      }
    } else {
#pragma unroll
      for (int k = 0; k < NR0; ++k) {
        const int x0 = F0::in_pos(k, jA);
        cpx<R> v = {R(0), R(0)};
        if (actA) v = gin[((long)x0 * L1 + x1A) * I + sA];
        if (a.apbc) v = mul_tw_rt<R, +1>(v, x0 * TWSTEP);
        x[k] = v;
      }
      if (idle) return;
    }
    if constexpr (MODE == P01_FWDCG) prefetch_next_tile();
    F0::run(x, jA);
    if constexpr (L1 == 1) {
      if (actA) {
#pragma unroll
        for (int k = 0; k < NR0; ++k) gout[(long)F0::out_pos(k, jA) * I + sA] = x[k];
      }
    } else {
      if (actA) {
#pragma unroll
        for (int k = 0; k < NR0; ++k) {
          const int n0 = F0::out_pos(k, jA);
          sm[n0 * PITCH0 + x1A * NSEG + sA] = x[k];
        }
      }
      __syncthreads();
      cpx<R> y[NR1];
#pragma unroll
      for (int k = 0; k < NR1; ++k) {
        cpx<R> v = {R(0), R(0)};
        if (actB) v = sm[x0B * PITCH0 + F1::in_pos(k, jB) * NSEG + sB];
        y[k] = v;
      }
      F1::run(y, jB);
      if (actB) {
#pragma unroll
        for (int k = 0; k < NR1; ++k)
          gout[((long)x0B * L1 + F1::out_pos(k, jB)) * I + sB] = y[k];
      }
    }
    if constexpr (MODE == P01_FWDCG && FIN == FIN_PP) {
      // shifted solves: <p,p> of this source for alpha = rho / (||M p||^2 + sigma <p,p>)
      const int blk = comp * gridDim.x + bx;
      if constexpr (p01_split_finalize<L0, L1>::v) block_partial(accp, a.red.for_source(src), blk, red_sh);  // k_finalize<FIN_PP> follows (launch_p01)
      else grid_reduce<FIN_PP>(accp, a.red.for_source(src), blk, 4 * gridDim.x, red_sh);
    }
  } else {
    // ---- inverse half: axis 1 first (from HBM), then axis 0 ----
    using G1 = LineFFT<R, L1, -1, VAR_DIT, TPL1>;
    using G0 = LineFFT<R, L0, -1, VAR_DIT, TPL0>;
    // operands of the site-local step (this thread's axis-0 line), one L2 prefetch hint per 32-byte sector
    auto prefetch_operands = [&]() {
      if constexpr (MODE != P01_INV) {
        if (actA && (sA * (int)sizeof(cpx<R>)) % 32 == 0) {
          const long fo = (long)f * V + i0;
#pragma unroll
          for (int k = 0; k < NR0; ++k) {
            const long off = ((long)G0::out_pos(k, jA) * L1 + x1A) * I + sA;
            prefetch_l2(as_stored<R, S>(a.psi) + (fo + off));
            prefetch_l2(a.phi + i0 + off);
            if constexpr (MODE == P01_ENDCG) prefetch_l2(s_r + (fo + off));
          }
        }
      }
    };
    cpx<R> x[NR0];
    if constexpr (L1 == 1) {
#pragma unroll
      for (int k = 0; k < NR0; ++k) {
        cpx<R> v = {R(0), R(0)};
        if (actA) v = gin[(long)G0::in_pos(k, jA) * I + sA];
        x[k] = v;
      }
      prefetch_operands();
    } else {
      {
        cpx<R> y[NR1];
#pragma unroll
        for (int k = 0; k < NR1; ++k) {
          cpx<R> v = {R(0), R(0)};
          if (actB) v = gin[((long)x0B * L1 + G1::in_pos(k, jB)) * I + sB];
          y[k] = v;
        }
        prefetch_operands();
        G1::run(y, jB);
        if (actB) {
#pragma unroll
          for (int k = 0; k < NR1; ++k) sm[x0B * PITCH0 + G1::out_pos(k, jB) * NSEG + sB] = y[k];
        }
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < NR0; ++k) {
        cpx<R> v = {R(0), R(0)};
        if (actA) v = sm[G0::in_pos(k, jA) * PITCH0 + x1A * NSEG + sA];
        x[k] = v;
      }
    }
    G0::run(x, jA);
    // post-twist exp(+i pi x0/T) and 1/V
#pragma unroll
    for (int k = 0; k < NR0; ++k) {
      const int x0 = G0::out_pos(k, jA);
      cpx<R> v = x[k];
      if (a.apbc) v = mul_tw_rt<R, -1>(v, x0 * TWSTEP);
      if constexpr (MODE == P01_INV) v = cscale(v, a.scale);  // the fused modes get 1/V from the multiply pass
      if constexpr (MODE == P01_ENDCG && sizeof(S) != sizeof(cpx<R>)) v = cscale(v, a.scale);  // binary16 storage: undo pass C's headroom factor
      x[k] = v;
    }
    if constexpr (MODE == P01_INV) {
      if (actA) {
#pragma unroll
        for (int k = 0; k < NR0; ++k)
          gout[((long)G0::out_pos(k, jA) * L1 + x1A) * I + sA] = x[k];
      }
    } else {
      // ---- site-local term of Eq. (2.19): + (m + 2 g phi) P+ psi + (m + 2 g phi)^* P- psi,
      //      spin 0,1 = P-, spin 2,3 = P+; M^dag swaps w and w^* ----
      // Preconditioned operator (op.pc): Mtilde = M M0^-1 = 1 + Y M0^-1 with
      // Y = 2 g phi P+ + 2 g^* phi^* P-, so the same passes serve with other site-local formulas:
      //   MID:  w = psi + Y t  (stored, ||w||^2),  then the forward half transforms Y^dag w (+ sigma t, Eq. 7.14);
      //   END / ENDCG:  q = t + w  (no phi).
      const bool use_conj = (comp < 2) != (a.op.dagger != 0);
      const bool pc = a.op.pc != 0;
      const bool pc_swap = pc && MODE == P01_MID;   // base = psi, multiplied = t
      const bool pc_unit = pc && MODE != P01_MID;   // coefficient 1
      const R m_re = pc ? R(0) : a.op.m_re, m_im = pc ? R(0) : a.op.m_im;
      const VP gpsi = as_stored<R, S>(a.psi) + ((long)f * V + i0);
      const cpx<R>* gphi = a.phi + i0;
      const VP gso = as_stored<R, S>(a.site_out) + ((long)f * V + i0);
      double acc = 0.0;
      constexpr int CH = (NR0 % 8 == 0) ? 8 : 4;  // sites whose operands are fetched together
      static_assert(NR0 % CH == 0, "chunking");
      if (actA) {
#pragma unroll
        for (int k0 = 0; k0 < NR0; k0 += CH) {
          long off[CH];
          cpx<R> ph[CH], ps[CH];
#pragma unroll
          for (int c = 0; c < CH; ++c) {
            off[c] = ((long)G0::out_pos(k0 + c, jA) * L1 + x1A) * I + sA;
            ph[c] = ldg_c(gphi + off[c]);
            if constexpr (MODE == P01_MID && !WZ_EVICT_MID) ps[c] = ldg_c(gpsi + off[c]);
            else ps[c] = ld_stream_nc(gpsi + off[c], pol);  // chi in pass E/E': read once, evict first
          }
          if constexpr (MODE == P01_ENDCG) {
            cpx<R> vr[CH];
            const VP gr = s_r + ((long)f * V + i0);
#pragma unroll
            for (int c = 0; c < CH; ++c) vr[c] = gr[off[c]];
            const R alpha = (R)a.red.st[src].alpha;
#pragma unroll
            for (int c = 0; c < CH; ++c) {
              cpx<R> w = {m_re + a.op.g2_re * ph[c].re - a.op.g2_im * ph[c].im,
                          m_im + a.op.g2_re * ph[c].im + a.op.g2_im * ph[c].re};
              if (use_conj) w.im = -w.im;
              if (pc_unit) w = {R(1), R(0)};
              cpx<R> q = x[k0 + c];
              q.re += w.re * ps[c].re - w.im * ps[c].im;
              q.im += w.re * ps[c].im + w.im * ps[c].re;
              if constexpr (FIN == FIN_RRS) {  // shifted system: q <- q + sigma p
                const cpx<R> vp = ldg_c(s_p + ((long)f * V + i0 + off[c]));
                q.re += a.op.shift * vp.re;
                q.im += a.op.shift * vp.im;
              }
              const cpx<R> rn = as_if_stored<R, S>({vr[c].re - alpha * q.re, vr[c].im - alpha * q.im});  // rho_k = ||r as stored||^2
              gr[off[c]] = rn;
              acc += (double)rn.re * (double)rn.re + (double)rn.im * (double)rn.im;
            }
          } else {
#pragma unroll
            for (int c = 0; c < CH; ++c) {
              cpx<R> w = {m_re + a.op.g2_re * ph[c].re - a.op.g2_im * ph[c].im,
                          m_im + a.op.g2_re * ph[c].im + a.op.g2_im * ph[c].re};
              if (use_conj) w.im = -w.im;
              if (pc_unit) w = {R(1), R(0)};
              const cpx<R> base = pc_swap ? ps[c] : x[k0 + c];
              const cpx<R> mul = pc_swap ? x[k0 + c] : ps[c];
              cpx<R> v = base;
              v.re += w.re * mul.re - w.im * mul.im;
              v.im += w.re * mul.im + w.im * mul.re;
              // value that enters the forward half (MID): v, or Y^dag v for the preconditioned operator;
              // preconditioned shifted system (Eq. 7.14): + sigma t with t = M0^-1 p, which
              // pass D turns into sigma (M0^-1)^dag M0^-1 p, and <p, A p> = ||w||^2 + sigma ||t||^2
              const cpx<R> tin = x[k0 + c];
              x[k0 + c] = pc_swap ? cpx<R>{w.re * v.re + w.im * v.im + a.op.shift * tin.re,
                                           w.re * v.im - w.im * v.re + a.op.shift * tin.im} : v;
              gso[off[c]] = v;
              if (FIN != FIN_STORE || a.red.partials) {
                acc += (double)v.re * (double)v.re + (double)v.im * (double)v.im;
                if (pc_swap) acc += (double)a.op.shift * ((double)tin.re * (double)tin.re + (double)tin.im * (double)tin.im);
              }
            }
          }
        }
      }
      if constexpr (MODE == P01_MID) {
        prefetch_next_tile();  // pass C: the forward half (about a quarter of the CTA's time) is left
        // forward again: pre-twist, DFT axis 0 (halves in -> DIF variant), DFT axis 1
        using F0 = LineFFT<R, L0, +1, VAR_DIF, TPL0>;
        using F1 = LineFFT<R, L1, +1, VAR_DIT, TPL1>;
        cpx<R> z[NR0];
#pragma unroll
        for (int k = 0; k < NR0; ++k) {
          const int x0 = G0::out_pos(k, jA);  // = out_index<NR0>(k) + jA*NR0 = F0::in_pos(oi(k), jA)
          cpx<R> v = x[k];
          if constexpr (sizeof(S) != sizeof(cpx<R>)) v = cscale(v, a.scale);  // binary16 storage: keeps the stored transform of chi in range
          if (a.apbc) v = mul_tw_rt<R, +1>(v, x0 * TWSTEP);
          z[out_index<NR0>(k)] = v;
        }
        F0::run(z, jA);
        if constexpr (L1 == 1) {
          if (actA) {
#pragma unroll
            for (int k = 0; k < NR0; ++k) gout[(long)F0::out_pos(k, jA) * I + sA] = z[k];
          }
        } else {
          __syncthreads();  // every axis-0 read of the tile is done
          if (actA) {
#pragma unroll
            for (int k = 0; k < NR0; ++k) sm[F0::out_pos(k, jA) * PITCH0 + x1A * NSEG + sA] = z[k];
          }
          __syncthreads();
          cpx<R> y[NR1];
#pragma unroll
          for (int k = 0; k < NR1; ++k) {
            cpx<R> v = {R(0), R(0)};
            if (actB) v = sm[x0B * PITCH0 + F1::in_pos(k, jB) * NSEG + sB];
            y[k] = v;
          }
          F1::run(y, jB);
          if (actB) {
#pragma unroll
            for (int k = 0; k < NR1; ++k)
              gout[((long)x0B * L1 + F1::out_pos(k, jB)) * I + sB] = y[k];
          }
        }
      }
      if (a.red.partials) {  // one reduction per source: its 4 spin components x all segments
        const int blk = comp * gridDim.x + bx;
        if constexpr (p01_split_finalize<L0, L1>::v) block_partial(acc, a.red.for_source(src), blk, red_sh);  // k_finalize<FIN> follows (launch_p01)
        else grid_reduce<FIN>(acc, a.red.for_source(src), blk, 4 * gridDim.x, red_sh);
      }
    }
  }
}

}  // namespace wz
