// wz_regfft.cuh -- 1D DFTs of compile-time length held in registers.
//
// Building block of the 4D FFT of PAPER.md:896-898 ("the crucial operation").
// One lattice line of length L (L = 2^a 3^b, L <= 64) is transformed by ONE thread
// (L/TPL = NR complex numbers in registers, TPL = 1) or by a PAIR of adjacent lanes
// (TPL = 2, one radix-2 step across the pair by warp shuffle).  Everything is fully
// unrolled: register indices, twiddle-table indices and the digit-reversed output
// order are compile-time constants, so the "bit reversal" costs nothing (the caller
// stores register k at position out_pos(k, j)).
//
// Transform convention (include/wz.h): DIR = +1 uses exp(-2 pi i n x / L)
// (forward), DIR = -1 uses exp(+2 pi i n x / L) (inverse, unnormalised here).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>

namespace wz {

template <typename R>
struct alignas(2 * sizeof(R)) cpx {
  R re, im;
};

// ---- storage types ---------------------------------------------------------------------
// Kernels compute in cpx<R>; vectors may be STORED narrower (NEXT-3): cpxh = one complex number as two
// IEEE binary16 values (4 bytes), converted on load / rounded to nearest even on store.  SPtr<R, S> is the pointer
// the kernels index: a raw cpx<R>* when S = cpx<R> (identical code to the untemplated kernels), a converting proxy
// otherwise.
struct alignas(4) cpxh {
  __half2 v;
};
template <typename R, typename S>
struct SRef {
  S* p;
  __device__ __forceinline__ operator cpx<R>() const {
    const float2 f = __half22float2(p->v);
    return {(R)f.x, (R)f.y};
  }
  __device__ __forceinline__ SRef& operator=(cpx<R> v) {
    p->v = __floats2half2_rn((float)v.re, (float)v.im);
    return *this;
  }
};
template <typename R, typename S>
struct SProxy {
  S* p;
  __device__ __forceinline__ SProxy operator+(long i) const { return {p + i}; }
  __device__ __forceinline__ SRef<R, S> operator[](long i) const { return {p + i}; }
  __device__ __forceinline__ const void* raw() const { return p; }
};
template <typename R, typename S> struct sptr { typedef SProxy<R, S> type; };
template <typename R> struct sptr<R, cpx<R>> { typedef cpx<R>* type; };
// the value a store to S-typed memory leaves there (identity when S = cpx<R>)
template <typename R, typename S>
__device__ __forceinline__ cpx<R> as_if_stored(cpx<R> v) {
  if constexpr (sizeof(S) == sizeof(cpx<R>)) return v;
  else {
    const float2 f = __half22float2(__floats2half2_rn((float)v.re, (float)v.im));
    return {(R)f.x, (R)f.y};
  }
}
// typed view of a base pointer the host passed as cpx<R>* (for narrower storage it points to S elements)
template <typename R, typename S>
__device__ __forceinline__ typename sptr<R, S>::type as_stored(const cpx<R>* base) {
  if constexpr (sizeof(S) == sizeof(cpx<R>)) return const_cast<cpx<R>*>(base);
  else return SProxy<R, S>{reinterpret_cast<S*>(const_cast<cpx<R>*>(base))};
}

// exp(-2 pi i j / TWN), j = 0..TWN-1.  384 = 2^7 * 3 covers every twiddle of the
// supported line lengths and the antiperiodic twist exp(-i pi x0 / T) (T | 192).
constexpr int TWN = 384;
// (private to each translation unit: every kernel module uploads its own copy, wz_kmod.cu)
static __constant__ float2 c_twf[TWN];
static __constant__ double2 c_twd[TWN];

template <typename R>
__device__ __forceinline__ cpx<R> tw_load(int idx);
template <>
__device__ __forceinline__ cpx<float> tw_load<float>(int idx) {
  float2 t = c_twf[idx];
  return {t.x, t.y};
}
template <>
__device__ __forceinline__ cpx<double> tw_load<double>(int idx) {
  double2 t = c_twd[idx];
  return {t.x, t.y};
}

template <typename R>
__device__ __forceinline__ cpx<R> cadd(cpx<R> a, cpx<R> b) { return {a.re + b.re, a.im + b.im}; }
template <typename R>
__device__ __forceinline__ cpx<R> csub(cpx<R> a, cpx<R> b) { return {a.re - b.re, a.im - b.im}; }
template <typename R>
__device__ __forceinline__ cpx<R> cmul(cpx<R> a, cpx<R> b) {
  return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re};
}
template <typename R>
__device__ __forceinline__ cpx<R> cconj(cpx<R> a) { return {a.re, -a.im}; }
template <typename R>
__device__ __forceinline__ cpx<R> cscale(cpx<R> a, R s) { return {a.re * s, a.im * s}; }
// multiply by -i*DIR  (DIR=+1: -i;  DIR=-1: +i)
template <typename R, int DIR>
__device__ __forceinline__ cpx<R> mul_mi(cpx<R> a) {
  if (DIR > 0) return {a.im, -a.re};
  return {-a.im, a.re};
}

// a * exp(-DIR 2 pi i num/den).  num, den are compile-time after unrolling, so the
// branches fold and the table index becomes a constant-bank immediate.
template <typename R, int DIR>
__device__ __forceinline__ cpx<R> mul_tw(cpx<R> a, int num, int den) {
  const int idx = (num % den) * (TWN / den);
  if (idx == 0) return a;
  if (idx == TWN / 4) return mul_mi<R, DIR>(a);
  if (idx == TWN / 2) return {-a.re, -a.im};
  if (idx == 3 * TWN / 4) return mul_mi<R, -DIR>(a);
  cpx<R> w = tw_load<R>(idx);
  if (DIR < 0) w.im = -w.im;
  return cmul(a, w);
}
// same with a run-time index (pair twiddles, twist)
template <typename R, int DIR>
__device__ __forceinline__ cpx<R> mul_tw_rt(cpx<R> a, int idx) {
  cpx<R> w = tw_load<R>(idx);
  if (DIR < 0) w.im = -w.im;
  return cmul(a, w);
}

// ---- packed FP32x2 (Blackwell FADD2/FFMA2): one instruction per complex add ----------
// A complex64 value is an aligned register pair, so a complex add/sub is ONE add.f32x2 /
// sub.f32x2 issue slot instead of two (same FP-pipe time, half the issue slots; the
// passes are issue-bound, profiles/r01_*).  Multiplications by twiddles stay scalar.
#define WZ_PACKED 1
__device__ __forceinline__ unsigned long long pk(cpx<float> a) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.re), "f"(a.im));
  return r;
}
__device__ __forceinline__ cpx<float> upk(unsigned long long v) {
  cpx<float> a;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(a.re), "=f"(a.im) : "l"(v));
  return a;
}
#if WZ_PACKED
template <>
__device__ __forceinline__ cpx<float> cadd<float>(cpx<float> a, cpx<float> b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)));
  return upk(r);
}
template <>
__device__ __forceinline__ cpx<float> csub<float>(cpx<float> a, cpx<float> b) {
  unsigned long long r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)));
  return upk(r);
}
#endif
// a + s * (b.im, -b.re) for s = +1 (a - i b) and the mirrored a + i b: one FFMA2 each
__device__ __forceinline__ cpx<float> fma_pm(cpx<float> bs /* (b.im, b.re) */, float c0, float c1, cpx<float> a) {
  unsigned long long r;
  cpx<float> c = {c0, c1};
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk(bs)), "l"(pk(c)), "l"(pk(a)));
  return upk(r);
}

// ---- small butterflies -------------------------------------------------------
template <typename R>
__device__ __forceinline__ void bf2(cpx<R>& a, cpx<R>& b) {
  cpx<R> t = csub(a, b);
  a = cadd(a, b);
  b = t;
}
template <typename R, int DIR>
__device__ __forceinline__ void bf4(cpx<R>& a, cpx<R>& b, cpx<R>& c, cpx<R>& d) {
  cpx<R> t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), t3 = mul_mi<R, DIR>(csub(b, d));
  a = cadd(t0, t2);
  c = csub(t0, t2);
  b = cadd(t1, t3);
  d = csub(t1, t3);
}
#if WZ_PACKED
template <int DIR>
__device__ __forceinline__ void bf4_packed(cpx<float>& a, cpx<float>& b, cpx<float>& c, cpx<float>& d) {
  const cpx<float> t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), u = csub(b, d);
  const cpx<float> us = {u.im, u.re};
  // forward: -i u = (u.im, -u.re);  inverse: +i u = (-u.im, u.re)
  const float s = (DIR > 0) ? 1.f : -1.f;
  a = cadd(t0, t2);
  c = csub(t0, t2);
  b = fma_pm(us, s, -s, t1);
  d = fma_pm(us, -s, s, t1);
}
#endif
template <typename R, int DIR>
__device__ __forceinline__ void bf3(cpx<R>& a, cpx<R>& b, cpx<R>& c) {
  const R h = R(0.86602540378443864676372317075294);  // sqrt(3)/2
  cpx<R> t = cadd(b, c);
  cpx<R> u = cscale(mul_mi<R, DIR>(csub(b, c)), h);
  cpx<R> mm = {a.re - R(0.5) * t.re, a.im - R(0.5) * t.im};
  a = cadd(a, t);
  b = cadd(mm, u);
  c = csub(mm, u);
}

template <int N>
struct radix_of {
  static constexpr int v = (N % 4 == 0) ? 4 : ((N % 2 == 0) ? 2 : 3);
};

// Position p of the in-place decimation-in-frequency result holds output index
// out_index<N>(p).
template <int N>
__host__ __device__ constexpr int out_index(int p) {
  if constexpr (N == 1) {
    return 0;
  } else {
    constexpr int r = radix_of<N>::v, m = N / r;
    return p / m + r * out_index<m>(p % m);
  }
}

// In-place DIF FFT of x[0..N-1] (registers).
template <typename R, int N, int DIR>
struct RegFFT {
  static __device__ __forceinline__ void run(cpx<R>* x) {
    if constexpr (N > 1) {
      constexpr int r = radix_of<N>::v, m = N / r;
#pragma unroll
      for (int k = 0; k < m; ++k) {
        if constexpr (r == 4) {
#if WZ_PACKED
          if constexpr (sizeof(R) == 4) bf4_packed<DIR>(x[k], x[k + m], x[k + 2 * m], x[k + 3 * m]);
          else
#endif
            bf4<R, DIR>(x[k], x[k + m], x[k + 2 * m], x[k + 3 * m]);
          x[k + m] = mul_tw<R, DIR>(x[k + m], k, N);
          x[k + 2 * m] = mul_tw<R, DIR>(x[k + 2 * m], 2 * k, N);
          x[k + 3 * m] = mul_tw<R, DIR>(x[k + 3 * m], 3 * k, N);
        } else if constexpr (r == 2) {
          bf2<R>(x[k], x[k + m]);
          x[k + m] = mul_tw<R, DIR>(x[k + m], k, N);
        } else {
          bf3<R, DIR>(x[k], x[k + m], x[k + 2 * m]);
          x[k + m] = mul_tw<R, DIR>(x[k + m], k, N);
          x[k + 2 * m] = mul_tw<R, DIR>(x[k + 2 * m], 2 * k, N);
        }
      }
#pragma unroll
      for (int q = 0; q < r; ++q) RegFFT<R, m, DIR>::run(x + q * m);
    }
  }
};

template <typename R>
__device__ __forceinline__ cpx<R> shfl_xor_c(cpx<R> v, int dist) {
  cpx<R> o;
  o.re = __shfl_xor_sync(0xffffffffu, v.re, dist);
  o.im = __shfl_xor_sync(0xffffffffu, v.im, dist);
  return o;
}

// Default lanes per line: at most 32 complex64 / 16 complex128 values per thread.
// (Kernels pick TPL per pass; more lanes per line = fewer registers, more warps.)
template <typename R, int L>
struct line_tpl {
  static constexpr int v = (L * (int)sizeof(R) > 128) ? 2 : 1;
};

// Thread -> (line, j) inside a group of threads working on lines with TPL lanes each:
// the G = 32/TPL lines of a warp sit in consecutive lanes (coalescing, bank-conflict
// free tiles), the lane sub-index j in the HIGH lane bits (shuffle distances G, 2G).
template <int TPL>
__device__ __forceinline__ void lane_split(int t, int& line, int& j) {
  constexpr int G = 32 / TPL;
  const int w = t >> 5, l = t & 31;
  line = w * G + (l % G);
  j = l / G;
}

enum { VAR_DIT = 0, VAR_DIF = 1 };

// One lattice line of length L handled by TPL lanes (1, 2 or 4); lane sub-index j,
// bit b of j <-> lane xor distance XD << b.  NR = L/TPL values per lane.
//  VAR_DIT: radix-2 steps across lanes AFTER the register FFT:
//           input  position of register k: 2*sub_in(k, j>>1) + (j&1)   (interleaved),
//           output index    of register k: sub_out(k, j>>1) + (j&1)*L/2 (blocks).
//  VAR_DIF: radix-2 steps across lanes BEFORE the register FFT: input in blocks,
//           output interleaved.  A DIT inverse feeds a DIF forward of the same TPL
//           without any cross-lane traffic (register k -> register out_index<NR>(k)).
// All 32 lanes of the warp must call run().
template <typename R, int L, int DIR, int VAR, int TPL, int XD = 32 / TPL>
struct LineFFT {
  static constexpr int NR = L / TPL;
  using Sub = LineFFT<R, L / 2, DIR, VAR, TPL / 2, XD * 2>;
  static __host__ __device__ constexpr int in_pos(int k, int j) {
    return (VAR == VAR_DIT) ? (2 * Sub::in_pos(k, j >> 1) + (j & 1)) : (Sub::in_pos(k, j >> 1) + (j & 1) * (L / 2));
  }
  static __host__ __device__ constexpr int out_pos(int k, int j) {
    return (VAR == VAR_DIT) ? (Sub::out_pos(k, j >> 1) + (j & 1) * (L / 2)) : (2 * Sub::out_pos(k, j >> 1) + (j & 1));
  }
  static __device__ __forceinline__ void run(cpx<R>* x, int j) {
    const bool odd = (j & 1) != 0;
    const R sgn = odd ? R(-1) : R(1);  // even lane: v + o, odd lane: o - v  ==  fma(sgn, v, o)
    if constexpr (VAR == VAR_DIT) {
      Sub::run(x, j >> 1);
      // twiddle w_L^n, n = Sub::out_pos(k, j>>1) = out_pos(k, 0) + lane part; the lane part
      // (TPL = 4 only) is L/4, i.e. a factor -i (forward) on the lanes with bit 1 of j set
#pragma unroll
      for (int k = 0; k < NR; ++k) {
        cpx<R> v = x[k];
        if (odd) {
          v = mul_tw<R, DIR>(v, Sub::out_pos(k, 0), L);
          if (TPL >= 4 && (j & 2)) v = mul_mi<R, DIR>(v);
        }
        cpx<R> o = shfl_xor_c(v, XD);
        x[k] = {fma(sgn, v.re, o.re), fma(sgn, v.im, o.im)};  // E + O' | E - O'
      }
    } else {
#pragma unroll
      for (int k = 0; k < NR; ++k) {
        cpx<R> v = x[k];
        cpx<R> o = shfl_xor_c(v, XD);
        cpx<R> t = {fma(sgn, v.re, o.re), fma(sgn, v.im, o.im)};  // lo + hi | lo - hi
        if (odd) {
          t = mul_tw<R, DIR>(t, Sub::in_pos(k, 0), L);
          if (TPL >= 4 && (j & 2)) t = mul_mi<R, DIR>(t);
        }
        x[k] = t;
      }
      Sub::run(x, j >> 1);
    }
  }
};
template <typename R, int L, int DIR, int VAR, int XD>
struct LineFFT<R, L, DIR, VAR, 1, XD> {
  static constexpr int NR = L;
  static __host__ __device__ constexpr int in_pos(int k, int) { return k; }
  static __host__ __device__ constexpr int out_pos(int k, int) { return out_index<L>(k); }
  static __device__ __forceinline__ void run(cpx<R>* x, int) { RegFFT<R, L, DIR>::run(x); }
};

}  // namespace wz
