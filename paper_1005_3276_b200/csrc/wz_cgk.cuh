// wz_cgk.cuh -- CG vector kernels:
// initialisation, the deferred x update, and the complex128 reliable-update pieces for complex64 solves (G9).
// Vectors are treated as flat real arrays of 2*4V entries, 16-byte accesses.
#pragma once
#include "wz_common.cuh"

namespace wz {

template <typename R>
struct vec16;
template <>
struct vec16<float> {
  typedef float4 T;
  static constexpr int N = 4;
};
template <>
struct vec16<double> {
  typedef double2 T;
  static constexpr int N = 2;
};

template <typename R>
__device__ __forceinline__ void ld16(const R* p, R (&v)[vec16<R>::N]) {
  typename vec16<R>::T t = *reinterpret_cast<const typename vec16<R>::T*>(p);
  const R* q = reinterpret_cast<const R*>(&t);
#pragma unroll
  for (int i = 0; i < vec16<R>::N; ++i) v[i] = q[i];
}
template <typename R>
__device__ __forceinline__ void st16(R* p, const R (&v)[vec16<R>::N]) {
  typename vec16<R>::T t;
  R* q = reinterpret_cast<R*>(&t);
#pragma unroll
  for (int i = 0; i < vec16<R>::N; ++i) q[i] = v[i];
  *reinterpret_cast<typename vec16<R>::T*>(p) = t;
}

constexpr int CGK_NT = 256;

// r = b, p = b (rounded to R if b is wider), xs = 0 (if given), X = 0 (complex128, if given);
// ||b||^2 (of the values as given) -> FIN_INIT.  TB: storage type of b.
template <typename R, typename TB>
__global__ void __launch_bounds__(CGK_NT)
k_cg_init(const TB* b, R* r, R* p /* b may alias r or p */, R* __restrict__ xs,
          double* __restrict__ X, long n, RedArgs red) {
  const int src = blockIdx.y;  // one source per grid row
  b += src * n; r += src * n; p += src * n;
  if (xs) xs += src * n;
  if (X) X += src * n;
  red = red.for_source(src);
  __shared__ double sh[33];
  double acc = 0.0;
  for (long i = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < n;
       i += (long)gridDim.x * blockDim.x * 2) {
    const TB b0 = b[i], b1 = b[i + 1];
    acc += (double)b0 * (double)b0 + (double)b1 * (double)b1;
    r[i] = (R)b0; r[i + 1] = (R)b1;
    p[i] = (R)b0; p[i + 1] = (R)b1;
    if (xs) { xs[i] = R(0); xs[i + 1] = R(0); }
    if (X) { X[i] = 0.0; X[i + 1] = 0.0; }
  }
  grid_reduce<FIN_INIT>(acc, red, blockIdx.x, gridDim.x, sh);
}

// sum |v|^2 -> FIN (one source per grid row)
template <typename TB, int FIN>
__global__ void __launch_bounds__(CGK_NT)
k_norm2(const TB* __restrict__ v, long n, RedArgs red) {
  v += blockIdx.y * n;
  red = red.for_source(blockIdx.y);
  __shared__ double sh[33];
  double acc = 0.0;
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x)
    acc += (double)v[i] * (double)v[i];
  grid_reduce<FIN>(acc, red, blockIdx.x, gridDim.x, sh);
}

// x += alpha p with the alpha still pending in the CG state (the fused pass A' applies
// it one iteration late); not gated.  k_clear_alpha then marks it as applied.
template <typename R>
__global__ void __launch_bounds__(CGK_NT)
k_flush_x(R* __restrict__ x, const R* __restrict__ p, long n, const CGState* st) {
  const int src = blockIdx.y;
  x += src * n; p += src * n; st += src;
  constexpr int N = vec16<R>::N;
  const R alpha = (R)st->alpha;
  if (alpha == R(0)) return;
  for (long i = ((long)blockIdx.x * blockDim.x + threadIdx.x) * N; i < n;
       i += (long)gridDim.x * blockDim.x * N) {
    R vx[N], vp[N];
    ld16<R>(x + i, vx);
    ld16<R>(p + i, vp);
#pragma unroll
    for (int e = 0; e < N; ++e) vx[e] = vx[e] + alpha * vp[e];
    st16<R>(x + i, vx);
  }
}
__global__ void k_clear_alpha(CGState* st) { st[blockIdx.x].alpha = 0.0; }

// Reliable update, part 1:  X += xs (complex128 += complex64);  xs = 0.
__global__ void __launch_bounds__(CGK_NT)
k_ru_accum(double* __restrict__ X, float* __restrict__ xs, long n) {
  X += blockIdx.y * n; xs += blockIdx.y * n;
  for (long i = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 4; i < n;
       i += (long)gridDim.x * blockDim.x * 4) {
    float v[4], z[4] = {0.f, 0.f, 0.f, 0.f};
    ld16<float>(xs + i, v);
    double2 a = *reinterpret_cast<double2*>(X + i), c = *reinterpret_cast<double2*>(X + i + 2);
    a.x += (double)v[0];
    a.y += (double)v[1];
    c.x += (double)v[2];
    c.y += (double)v[3];
    *reinterpret_cast<double2*>(X + i) = a;
    *reinterpret_cast<double2*>(X + i + 2) = c;
    st16<float>(xs + i, z);
  }
}

// Residual in float64:  d = b - q - sigma x  (sigma x only if xshift is given);  sum |d|^2 -> FIN;
// r = round(d) (if r given).  TB: storage type of b, TR: storage type of r.
template <typename TB, typename TR, int FIN>
__global__ void __launch_bounds__(CGK_NT)
k_resid(const TB* __restrict__ b, const double* __restrict__ q, TR* __restrict__ r, long n,
        RedArgs red, const double* __restrict__ xshift = nullptr, double sigma = 0.0) {
  const int src = blockIdx.y;
  b += src * n; q += src * n;
  if (r) r += src * n;
  if (xshift) xshift += src * n;
  red = red.for_source(src);
  __shared__ double sh[33];
  double acc = 0.0;
  for (long i = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < n;
       i += (long)gridDim.x * blockDim.x * 2) {
    double2 vq = *reinterpret_cast<const double2*>(q + i);
    double d0 = (double)b[i] - vq.x, d1 = (double)b[i + 1] - vq.y;
    if (xshift) {
      d0 -= sigma * xshift[i];
      d1 -= sigma * xshift[i + 1];
    }
    acc += d0 * d0 + d1 * d1;
    if (r) {
      r[i] = (TR)d0;
      r[i + 1] = (TR)d1;
    }
  }
  grid_reduce<FIN>(acc, red, blockIdx.x, gridDim.x, sh);
}

// Rational sum, Eq. (7.6):  out = alpha_0 eta  (first = 1)  or  out += alpha_i X_i,
// complex128 accumulation; one source per grid row.  TB: storage type of the term.
template <typename TB>
__global__ void __launch_bounds__(CGK_NT)
k_rat_term(double* __restrict__ out, const TB* __restrict__ v, double a, long n, int first) {
  out += blockIdx.y * n; v += blockIdx.y * n;
  for (long i = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < n;
       i += (long)gridDim.x * blockDim.x * 2) {
    double2 o = first ? make_double2(0.0, 0.0) : *reinterpret_cast<double2*>(out + i);
    o.x += a * (double)v[i];
    o.y += a * (double)v[i + 1];
    *reinterpret_cast<double2*>(out + i) = o;
  }
}

// Locality probe, Eq. (3.10)-(3.11):  f(r) = max{ ||psi(x)|| : ||x||_1 = r } with
// the taxi-driver distance to the origin (shorter way round each axis) and ||.|| the norm over
// the four spin components.  f holds ||.||^2 as the bit pattern of a non-negative double, so
// an unsigned 64-bit atomicMax orders it; the host takes the square root.
template <typename R>
__global__ void __launch_bounds__(CGK_NT)
k_locality(const cpx<R>* __restrict__ psi, unsigned long long* __restrict__ f, int L0, int L1, int L2, int L3) {
  const long V = (long)L0 * L1 * L2 * L3;
  for (long x = (long)blockIdx.x * blockDim.x + threadIdx.x; x < V; x += (long)gridDim.x * blockDim.x) {
    double n2 = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const cpx<R> v = psi[c * V + x];
      n2 += (double)v.re * (double)v.re + (double)v.im * (double)v.im;
    }
    long t = x;
    const int x3 = (int)(t % L3); t /= L3;
    const int x2 = (int)(t % L2); t /= L2;
    const int x1 = (int)(t % L1); t /= L1;
    const int x0 = (int)t;
    const int r = min(x0, L0 - x0) + min(x1, L1 - x1) + min(x2, L2 - x2) + min(x3, L3 - x3);
    atomicMax(f + r, (unsigned long long)__double_as_longlong(n2));
  }
}


// ---- multi-shift CG (Eq. 7.6-7.7, 927-931 Eq. 7.13) ----------------
// All systems (A + sigma_i) x_i = b from the Krylov space of ONE CG iteration (the base system, the smallest
// shift): the residual of shift i stays collinear with the base residual, r_i = zeta_i r (B. Jegerlehner,
// hep-lat/9612014).  Per base iteration n (alpha_n, beta_n the base CG coefficients, s_i = sigma_i - sigma_base):
//   zeta_{n+1} = zeta_n zeta_{n-1} alpha_{n-1} / (alpha_n beta_{n-1} (zeta_{n-1} - zeta_n) + zeta_{n-1} alpha_{n-1} (1 + s_i alpha_n))
//   x_i += alpha_n (zeta_{n+1}/zeta_n) p_i;   p_i = zeta_{n+1} r_{n+1} + beta_n (zeta_{n+1}/zeta_n)^2 p_i
// A shift is frozen once |zeta| ||r|| <= tol ||b||.
constexpr int WZ_MAX_SHIFTS = 32;
struct MSState {  // per source
  double zeta[WZ_MAX_SHIFTS], zeta_prev[WZ_MAX_SHIFTS];
  double ax[WZ_MAX_SHIFTS];    // coefficient of p_i in this iteration's x_i update
  double zr[WZ_MAX_SHIFTS];    // coefficient of r in this iteration's p_i update
  double bp[WZ_MAX_SHIFTS];    // coefficient of p_i in this iteration's p_i update
  double rec[WZ_MAX_SHIFTS];   // |zeta| ||r|| / ||b|| at the shift's last update
  double srel[WZ_MAX_SHIFTS];  // sigma_i - sigma_base
  double alpha_prev, beta_prev;
  int upd[WZ_MAX_SHIFTS];      // 1: the vectors of shift i take part in this iteration's update
  int frozen[WZ_MAX_SHIFTS];
  int its[WZ_MAX_SHIFTS];      // base iteration of the shift's last update
  int nshift, last_iter;
};

// One thread per source, after pass E' of the base iteration: the scalar recurrences.
__global__ void k_ms_scalars(MSState* ms_, const CGState* st_) {
  MSState* ms = ms_ + blockIdx.x;
  const CGState* st = st_ + blockIdx.x;
  const int i = threadIdx.x;
  if (i >= ms->nshift) return;
  const bool advanced = st->iter != ms->last_iter;  // the base took a step since the last call
  int upd = 0;
  if (advanced && !ms->frozen[i]) {
    const double alpha = st->alpha, beta = st->beta;
    const double zn = ms->zeta[i], zp = ms->zeta_prev[i];
    const double znew = zn * zp * ms->alpha_prev /
                        (alpha * ms->beta_prev * (zp - zn) + zp * ms->alpha_prev * (1.0 + ms->srel[i] * alpha));
    const double ratio = znew / zn;
    ms->ax[i] = alpha * ratio;
    ms->zr[i] = znew;
    ms->bp[i] = beta * ratio * ratio;
    ms->zeta_prev[i] = zn;
    ms->zeta[i] = znew;
    ms->its[i] = st->iter;
    const double rn = fabs(znew) * sqrt(st->rr);
    ms->rec[i] = st->bnorm > 0.0 ? rn / st->bnorm : 0.0;
    if (rn <= st->tol * st->bnorm) ms->frozen[i] = 1;
    upd = 1;
  }
  ms->upd[i] = upd;
  __syncthreads();
  if (i == 0 && advanced) {
    ms->alpha_prev = st->alpha;
    ms->beta_prev = st->beta;
    ms->last_iter = st->iter;
  }
}

// x_i += ax_i p_i;  p_i = zr_i r + bp_i p_i  for every shift that takes part (upd), r read once per element.
// Vectors: [shift][source][n] for ps and xsh; r: [source][n].  TX: storage type of the x_i.
template <typename R, typename TX>
__global__ void __launch_bounds__(CGK_NT)
k_ms_update(const R* __restrict__ r, R* __restrict__ ps, TX* __restrict__ xsh, long n, int nb, int base,
            const MSState* __restrict__ ms_) {
  const int src = blockIdx.y;
  const MSState* ms = ms_ + src;
  __shared__ double s_ax[WZ_MAX_SHIFTS], s_zr[WZ_MAX_SHIFTS], s_bp[WZ_MAX_SHIFTS];
  __shared__ int s_upd[WZ_MAX_SHIFTS];
  const int ns = ms->nshift;
  if (threadIdx.x < ns) {
    s_ax[threadIdx.x] = ms->ax[threadIdx.x]; s_zr[threadIdx.x] = ms->zr[threadIdx.x];
    s_bp[threadIdx.x] = ms->bp[threadIdx.x];
    s_upd[threadIdx.x] = (threadIdx.x == base) ? 0 : ms->upd[threadIdx.x];  // the base system is advanced by passes A'/E'
  }
  __syncthreads();
  bool any = false;
  for (int i = 0; i < ns; ++i) any |= (s_upd[i] != 0);
  if (!any) return;
  r += src * n;
  for (long e = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 2; e < n; e += (long)gridDim.x * blockDim.x * 2) {
    const R r0 = r[e], r1 = r[e + 1];
    for (int i = 0; i < ns; ++i) {
      if (!s_upd[i]) continue;
      const size_t o = ((size_t)i * nb + src) * n + e;
      const R p0 = ps[o], p1 = ps[o + 1];
      xsh[o] = (TX)((double)xsh[o] + s_ax[i] * (double)p0);
      xsh[o + 1] = (TX)((double)xsh[o + 1] + s_ax[i] * (double)p1);
      ps[o] = (R)(s_zr[i] * (double)r0 + s_bp[i] * (double)p0);
      ps[o + 1] = (R)(s_zr[i] * (double)r1 + s_bp[i] * (double)p1);
    }
  }
}

// ps_i = b, x_i = 0 for every shift (one source per grid row, all shifts).  TB: storage type of b.
template <typename R, typename TX, typename TB>
__global__ void __launch_bounds__(CGK_NT)
k_ms_init(const TB* __restrict__ b, R* __restrict__ ps, TX* __restrict__ xsh, long n, int nb, int ns) {
  const int src = blockIdx.y;
  b += src * n;
  for (long e = (long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long)gridDim.x * blockDim.x) {
    const R v = (R)b[e];
    for (int i = 0; i < ns; ++i) {
      const size_t o = ((size_t)i * nb + src) * n + e;
      ps[o] = v;
      xsh[o] = TX(0);
    }
  }
}

// ---- binary16 storage of the inner solver's vectors (wz_cg_solve_dc_half; oracle O10) ----------
// r = p = binary16(s d) for the float defect d and the normalisation s (unit rms), x = 0 (float);
// sum |r|^2 of the values AS STORED -> FIN_INIT.  One source per launch.
__global__ void __launch_bounds__(CGK_NT)
k_h_init(const float* __restrict__ d, __half* __restrict__ r, __half* __restrict__ p, float* __restrict__ x, long n,
         double s, RedArgs red) {
  __shared__ double sh[33];
  double acc = 0.0;
  for (long i = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < n; i += (long)gridDim.x * blockDim.x * 2) {
    const __half2 h = __floats2half2_rn((float)(s * (double)d[i]), (float)(s * (double)d[i + 1]));
    *reinterpret_cast<__half2*>(r + i) = h;
    *reinterpret_cast<__half2*>(p + i) = h;
    x[i] = 0.f; x[i + 1] = 0.f;
    const float2 f = __half22float2(h);
    acc += (double)f.x * (double)f.x + (double)f.y * (double)f.y;
  }
  grid_reduce<FIN_INIT>(acc, red, blockIdx.x, gridDim.x, sh);
}

// x (float) += alpha p (binary16) with the alpha still pending in the CG state (see k_flush_x); one source per grid row.
__global__ void __launch_bounds__(CGK_NT)
k_h_flush_x(float* __restrict__ x, const __half* __restrict__ p, long n, const CGState* st) {
  const int src = blockIdx.y;
  x += src * n; p += src * n; st += src;
  const float alpha = (float)st->alpha;
  if (alpha == 0.f) return;
  for (long i = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < n; i += (long)gridDim.x * blockDim.x * 2) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(p + i));
    x[i] += alpha * f.x;
    x[i + 1] += alpha * f.y;
  }
}

// X (complex128) += e (float) / s: the correction of one outer step, back in the units of the original system.
__global__ void __launch_bounds__(CGK_NT)
k_h_accum(double* __restrict__ X, const float* __restrict__ e, long n, double inv_s) {
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x)
    X[i] += inv_s * (double)e[i];
}

// Reliable update of the binary16-storage solver: r = binary16(s' d) for the recomputed float defect d, p = binary16(f p)
// (both back at unit rms); sum |r|^2 as stored -> FIN_HRU.  One source per launch.
__global__ void __launch_bounds__(CGK_NT)
k_h_rescale(const float* __restrict__ d, __half* __restrict__ r, __half* __restrict__ p, long n, double s_new, float f,
            RedArgs red) {
  __shared__ double sh[33];
  double acc = 0.0;
  for (long i = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < n; i += (long)gridDim.x * blockDim.x * 2) {
    const __half2 h = __floats2half2_rn((float)(s_new * (double)d[i]), (float)(s_new * (double)d[i + 1]));
    *reinterpret_cast<__half2*>(r + i) = h;
    const float2 pv = __half22float2(*reinterpret_cast<const __half2*>(p + i));
    *reinterpret_cast<__half2*>(p + i) = __floats2half2_rn(f * pv.x, f * pv.y);
    const float2 g = __half22float2(h);
    acc += (double)g.x * (double)g.x + (double)g.y * (double)g.y;
  }
  grid_reduce<FIN_HRU>(acc, red, blockIdx.x, gridDim.x, sh);
}
// what FIN_HRU needs (f^2, the new scaled ||b||), or: the update found the true residual below tol
__global__ void k_h_patch(CGState* st, double f2, double bnorm_scaled, int converged) {
  st->aux = f2;
  st->pp = bnorm_scaled;
  if (converged) { st->converged = 1; st->need_ru = 0; st->n_ru += 1; }
}
// X (complex128) += x (float) / s;  x = 0
__global__ void __launch_bounds__(CGK_NT)
k_h_accum_clear(double* __restrict__ X, float* __restrict__ x, long n, double inv_s) {
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
    X[i] += inv_s * (double)x[i];
    x[i] = 0.f;
  }
}

// dst (double) = src (TX) element-wise, or dst += src
template <typename TX>
__global__ void __launch_bounds__(CGK_NT)
k_to_double(double* __restrict__ dst, const TX* __restrict__ src, long n, int accumulate) {
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x)
    dst[i] = (accumulate ? dst[i] : 0.0) + (double)src[i];
}

// dst (double) = src (float), element-wise (phi for the complex128 operator of a
// complex64 plan: the float-rounded values, exactly what the oracle consumes).
__global__ void __launch_bounds__(CGK_NT)
k_f2d(double* __restrict__ dst, const float* __restrict__ src, long n) {
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (long)gridDim.x * blockDim.x)
    dst[i] = (double)src[i];
}

}  // namespace wz
