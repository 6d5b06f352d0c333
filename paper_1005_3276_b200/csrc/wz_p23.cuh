// wz_p23.cuh -- the contiguous two-axis pass: DFTs over axes (x2, x3) of the four
// spin components of one (n0, n1) plane, with the momentum-diagonal overlap
// multiply between the forward and the inverse half (SURVEY 7.2 passes B, D;
// step a3 of SURVEY 8(a)).
//
// Momentum-space operator (Eq. 2.19-2.20; 210-225 Eq. 3.1, 3.3;
// 382-390 Eq. 4.1-4.2; readings G1-G3 of DESIGN.md):
//   Dslash(p) = i c(p) sum_mu gamma_mu sin p_mu,   c = 2 rho / (s + Mw),
//   Mw = rho - 2 sum_mu sin^2(p_mu/2),  s = sqrt(Mw^2 + sum_mu sin^2 p_mu),
// with the gammas of Eq. (2.2), i.e. in 2x2 blocks
//   Dslash = i c [[0, B], [B^dag, 0]],  B = sin p0 + i sigma_k sin p_k.
// For Mw < 0 the cancellation-free form c = 2 rho (s - Mw) / sum sin^2 is used.
#pragma once
#include "wz_common.cuh"

namespace wz {

enum { P23_FFT = 0, P23_MULT = 1, P23_MULTPC = 2 };  // MULTPC: the multiply with args.pc = 1 or 2
// Preconditioner (Eq. 7.11): with args.pc set, the multiply applies the free
// inverse  M0^-1(p) = (-i c gamma.sin p + m^* P+ + m P-) / (c^2 sum sin^2 p + |m|^2)  (pc = 1) or its
// conjugate transpose M0(p) / (...) (pc = 2) instead of +-Dslash(p): same off-diagonal 2x2 blocks
// scaled by -+c/D, plus the diagonal m/D, m^*/D on the thread's own component.

// c(p) = k / (s + Mw) with s = sqrt(Mw^2 + S2), k = 2 rho sign / V; for Mw < 0 the
// cancellation-free form k (s - Mw) / S2 = k (s + |Mw|) / S2.  float: rsqrt/rcp approximations
// (<= 2 ulp each, far inside the 2e-5 matvec tolerance); double: IEEE sqrt and divide.
__device__ __forceinline__ float overlap_c(float Mw, float S2, float k) {
  const float q = fmaf(Mw, Mw, S2);
  const float a = fmaf(q, rsqrtf(q), fabsf(Mw));  // s + |Mw|: no cancellation on either branch
  const bool pos = Mw >= 0.f;
  return __fdividef(pos ? k : k * a, pos ? a : S2);
}
__device__ __forceinline__ double overlap_c(double Mw, double S2, double k) {
  const double a = sqrt(Mw * Mw + S2) + fabs(Mw);
  return (Mw >= 0.0) ? k / a : k * a / S2;
}

template <typename R>
struct P23Args {
  const cpx<R>* in;   // [nb][4][L0*L1][L2][L3]
  cpx<R>* out;        // may alias in
  int nplanes;        // L0*L1
  int L1;             // to split the plane index into (n0, n1)
  R scale;            // applied at the final store
  const R* tab;       // momentum tables [2][4][64]: sin p_mu(n), sin^2(p_mu(n)/2)
  R rho;
  R sign;             // +1: Dslash, -1: Dslash^dag = -Dslash
  int pc;             // 0: Dslash;  1: M0^-1;  2: (M0^-1)^dag
  R m_re, m_im;       // m (pc only)
  const CGState* gate;  // [nbatch], indexed by blockIdx.y
  int rev;              // 1: CTAs take (plane, source) in reverse order (L2 reuse across launches)
  int pf_dist;          // > 0: L2-prefetch the planes of the CTA pf_dist launches-in-order ahead (one wave)
};

// NC = spin components per CTA: 4 (whole plane quad, in place), or 2 when four planes
// do not fit in shared memory (64x64 complex128).  With NC = 2 the CTA with
// blockIdx.z = h reads components (2,3) [h = 0] or (0,1) [h = 1] and, for the multiply,
// writes the OTHER pair -- so in != out is required there (ping-pong buffers).
template <typename R, int L2, int L3, int T2, int T3, int NC = 4>
struct P23Cfg {
  static constexpr int TPL2 = T2, TPL3 = T3;  // lanes per line along axis 2 / axis 3
  static constexpr int NR2 = L2 / TPL2, NR3 = L3 / TPL3;
  static constexpr int NTC_A = L3 * TPL2;  // threads per component, lines along axis 2
  static constexpr int NTC_B = L2 * TPL3;  // lines along axis 3
  static constexpr int NTC_RAW = NTC_A > NTC_B ? NTC_A : NTC_B;
  static constexpr int NTC = (NTC_RAW + 31) / 32 * 32;  // whole warps per spin component
  static constexpr int NT = NC * NTC;
  static constexpr int PITCH = L3 + 1;            // row pitch (elements)
  static constexpr int CPITCH = L2 * PITCH + 4;   // component pitch
  static constexpr int CF_ELEMS = L2 * PITCH;  // per-site factor(s) of the multiply, computed once, shared by the components
  static constexpr size_t SMEM = sizeof(cpx<R>) * NC * (size_t)CPITCH + sizeof(R) * CF_ELEMS;
  static constexpr size_t SMEM_PC = SMEM + sizeof(R) * CF_ELEMS;  // + the diagonal factor (launches with args.pc)
};

template <typename R, int L2, int L3, int T2, int T3, int MODE, int DIR, int NC = 4>
__global__ void __launch_bounds__(P23Cfg<R, L2, L3, T2, T3, NC>::NT)
k_p23(const P23Args<R> a) {
  using Cfg = P23Cfg<R, L2, L3, T2, T3, NC>;
  constexpr int TPL2 = Cfg::TPL2, TPL3 = Cfg::TPL3, NR2 = Cfg::NR2, NR3 = Cfg::NR3;
  constexpr int NTC = Cfg::NTC, PITCH = Cfg::PITCH, CPITCH = Cfg::CPITCH;
  constexpr bool kMult = (MODE == P23_MULT || MODE == P23_MULTPC);
  constexpr bool kPC = (MODE == P23_MULTPC);
  constexpr int D1 = kMult ? +1 : DIR;  // direction of the first half
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cpx<R>* sm = reinterpret_cast<cpx<R>*>(smem_raw);
  R* cfs = reinterpret_cast<R*>(sm + NC * CPITCH);  // off-diagonal factor
  R* dgs = cfs + Cfg::CF_ELEMS;                     // diagonal factor (pc launches only)
  __shared__ R tb[2 * 4 * 64];

  const int bxr = a.rev ? (int)(gridDim.x - 1 - blockIdx.x) : (int)blockIdx.x;
  const int byr = a.rev ? (int)(gridDim.y - 1 - blockIdx.y) : (int)blockIdx.y;
  if (a.gate && !cg_active(a.gate + byr)) return;

  const int tid = threadIdx.x;
  const int plane = bxr;
  const long PL = (long)L2 * L3;
  const long fbase = (long)byr * 4 * a.nplanes;  // first field of this batch entry

  if constexpr (kMult) {
    for (int i = tid; i < 2 * 4 * 64; i += blockDim.x) tb[i] = a.tab[i];
  }

  const int cl = tid / NTC;     // component slot in this CTA (NTC is a multiple of 32)
  const int tc = tid % NTC;
  // global spin component read (cin) and written (cc) by this thread
  const int half = (NC == 4) ? 0 : (int)blockIdx.z;
  const int cin = (NC == 4) ? cl : (kMult ? (half ? cl : 2 + cl) : 2 * half + cl);
  const int cc = (NC == 4) ? cl : (kMult ? (half ? 2 + cl : cl) : 2 * half + cl);
  // role A: line along axis 2 at x3;  role B: line along axis 3 at n2
  int x3A, jA, n2B, jB;
  lane_split<TPL2>(tc, x3A, jA);
  lane_split<TPL3>(tc, n2B, jB);
  const bool actA = x3A < L3;
  const bool actB = n2B < L2;
  const cpx<R>* gin = a.in + (fbase + (long)cin * a.nplanes + plane) * PL;
  cpx<R>* gout = a.out + (fbase + (long)cc * a.nplanes + plane) * PL;
  cpx<R>* smc = sm + cl * CPITCH;

  // ---- half 1, axis 2 (lanes run along x3: coalesced HBM reads) ----
  {
    using F2 = LineFFT<R, L2, D1, VAR_DIT, TPL2>;
    cpx<R> x[NR2];
#pragma unroll
    for (int k = 0; k < NR2; ++k) {
      cpx<R> v = {R(0), R(0)};
      if (actA) v = gin[(long)F2::in_pos(k, jA) * L3 + x3A];
      x[k] = v;
    }
    // next wave's planes -> L2 while this CTA computes (one bulk prefetch per spin plane): the CTA that
    // takes them later pays L2 latency instead of HBM latency (the pass is latency-bound, profiles/r01_*)
    if constexpr (NC == 4) {
      if (a.pf_dist > 0 && tid < 4) {
        const long lin = (long)blockIdx.y * gridDim.x + blockIdx.x + a.pf_dist;
        if (lin < (long)gridDim.y * gridDim.x) {
          long by = lin / gridDim.x, bx = lin % gridDim.x;  // launch order -> data order
          if (a.rev) { by = gridDim.y - 1 - by; bx = gridDim.x - 1 - bx; }
          const cpx<R>* pf = a.in + ((by * 4 + tid) * a.nplanes + bx) * PL;
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(pf), "r"((unsigned)(PL * sizeof(cpx<R>))));
        }
      }
    }
    F2::run(x, jA);
    if (actA) {
#pragma unroll
      for (int k = 0; k < NR2; ++k) smc[F2::out_pos(k, jA) * PITCH + x3A] = x[k];
    }
  }
  __syncthreads();
  // ---- half 1, axis 3 ----
  {
    using F3 = LineFFT<R, L3, D1, VAR_DIT, TPL3>;
    cpx<R> y[NR3];
#pragma unroll
    for (int k = 0; k < NR3; ++k) {
      cpx<R> v = {R(0), R(0)};
      if (actB) v = smc[n2B * PITCH + F3::in_pos(k, jB)];
      y[k] = v;
    }
    F3::run(y, jB);
    if constexpr (kMult) {
      // c(p) once per momentum site: component slot cl covers 1/NC of this lane's n3 values
      static_assert(NR3 % NC == 0, "c(p) sharing");
      if (actB) {
        using G3i = LineFFT<R, L3, -1, VAR_DIF, TPL3>;
        const int n0 = plane / a.L1, n1 = plane % a.L1;
        const R* sn = tb;
        const R* sh = tb + 4 * 64;
        const R s0 = sn[0 * 64 + n0], s1 = sn[1 * 64 + n1], s2 = sn[2 * 64 + n2B];
        const R S012 = s0 * s0 + s1 * s1 + s2 * s2;
        const R Mw012 = a.rho - R(2) * (sh[0 * 64 + n0] + sh[1 * 64 + n1] + sh[2 * 64 + n2B]);
        const R kk = R(2) * a.rho * a.sign * a.scale;  // 1/V of the inverse transform rides along
#pragma unroll
        for (int k = cl * (NR3 / NC); k < (cl + 1) * (NR3 / NC); ++k) {
          const int n3 = G3i::in_pos(k, jB);
          const R s3 = sn[3 * 64 + n3];
          const R S2 = S012 + s3 * s3;
          const R cf = overlap_c(Mw012 - R(2) * sh[3 * 64 + n3], S2, kk);
          if constexpr (kPC) {  // cf carries rho-scaling and 1/V; c = cf / a.scale;  D = c^2 S2 + |m|^2
            const R c = cf / a.scale;
            const R invD = R(1) / (c * c * S2 + a.m_re * a.m_re + a.m_im * a.m_im);
            cfs[n2B * PITCH + n3] = cf * invD;
            dgs[n2B * PITCH + n3] = a.scale * invD;
          } else {
            cfs[n2B * PITCH + n3] = cf;
          }
        }
      }
    }
    __syncthreads();  // pair partners have read their half of the row
    if (actB) {
#pragma unroll
      for (int k = 0; k < NR3; ++k) smc[n2B * PITCH + F3::out_pos(k, jB)] = y[k];
    }
  }
  __syncthreads();

  if constexpr (MODE == P23_FFT) {
    // coalesced copy-out of the four planes
    for (int i = tid; i < NC * L2 * L3; i += blockDim.x) {
      const int ci = i / (L2 * L3), r = i % (L2 * L3);
      const int n2 = r / L3, n3 = r % L3;
      cpx<R> v = sm[ci * CPITCH + n2 * PITCH + n3];
      const int cg = (NC == 4) ? ci : 2 * half + ci;
      a.out[(fbase + (long)cg * a.nplanes + plane) * PL + r] = cscale(v, a.scale);
    }
  } else {
    // ---- momentum-diagonal multiply, then inverse axis 3 ----
    using G3 = LineFFT<R, L3, -1, VAR_DIF, TPL3>;
    using G2 = LineFFT<R, L2, -1, VAR_DIT, TPL2>;
    cpx<R> y[NR3];
    {
      const int n0 = plane / a.L1, n1 = plane % a.L1;
      const R* sn = tb;             // sin p_mu
      const R* sh = tb + 4 * 64;    // sin^2(p_mu/2)
      const int n2 = actB ? n2B : 0;
      const R s0 = sn[0 * 64 + n0], s1 = sn[1 * 64 + n1], s2 = sn[2 * 64 + n2];
      // out_c = i c(p) sign (Ca psi_ca + Cb psi_cb),  Ca = (A0, A1 + A3 s3), Cb = (B0, B1 + B3 s3)
      R A0, A1, A3, B0, B1, B3;
      if (cc == 0)      { A0 = s0;  A1 = R(0); A3 = R(1);  B0 = s2;  B1 = s1;   B3 = R(0); }
      else if (cc == 1) { A0 = -s2; A1 = s1;   A3 = R(0);  B0 = s0;  B1 = R(0); B3 = R(-1); }
      else if (cc == 2) { A0 = s0;  A1 = R(0); A3 = R(-1); B0 = -s2; B1 = -s1;  B3 = R(0); }
      else              { A0 = s2;  A1 = -s1;  A3 = R(0);  B0 = s0;  B1 = R(0); B3 = R(1); }
      // pc = 1 (M0^-1): upper components carry m, lower m^*;  pc = 2 (dagger): the other way round
      const R dm_re = a.m_re;
      const R dm_im = ((cc < 2) == (a.pc == 1)) ? a.m_im : -a.m_im;
      // inputs of output component cc: (psi_2, psi_3) for cc < 2, (psi_0, psi_1) otherwise;
      // with NC = 2 those are the two planes this CTA holds
      const cpx<R>* sa = sm + ((NC == 4) ? ((cc < 2) ? 2 : 0) : 0) * CPITCH + n2 * PITCH;
      const cpx<R>* sb = sa + CPITCH;
#pragma unroll
      for (int k = 0; k < NR3; ++k) {
        const int n3 = G3::in_pos(k, jB);
        const R s3 = sn[3 * 64 + n3];
        const R cf = cfs[n2 * PITCH + n3];
        const cpx<R> pa = sa[n3], pb = sb[n3];
        const R Ai = A1 + A3 * s3, Bi = B1 + B3 * s3;
        const R tr = A0 * pa.re - Ai * pa.im + B0 * pb.re - Bi * pb.im;
        const R ti = A0 * pa.im + Ai * pa.re + B0 * pb.im + Bi * pb.re;
        cpx<R> o = {-cf * ti, cf * tr};  // times i
        if constexpr (kPC) {  // + (m or m^*) / D on the own component
          const cpx<R> own = smc[n2 * PITCH + n3];
          const R dg = dgs[n2 * PITCH + n3];
          const R dr = dm_re * dg, di = dm_im * dg;
          o.re += dr * own.re - di * own.im;
          o.im += dr * own.im + di * own.re;
        }
        y[k] = o;
      }
    }
    G3::run(y, jB);
    __syncthreads();  // all momentum-space reads done
    if (actB) {
#pragma unroll
      for (int k = 0; k < NR3; ++k) smc[n2B * PITCH + G3::out_pos(k, jB)] = y[k];
    }
    __syncthreads();
    // ---- inverse axis 2, coalesced HBM writes ----
    cpx<R> x[NR2];
#pragma unroll
    for (int k = 0; k < NR2; ++k) {
      cpx<R> v = {R(0), R(0)};
      if (actA) v = smc[G2::in_pos(k, jA) * PITCH + x3A];
      x[k] = v;
    }
    G2::run(x, jA);
    if (actA) {
#pragma unroll
      for (int k = 0; k < NR2; ++k)
        gout[(long)G2::out_pos(k, jA) * L3 + x3A] = x[k];
    }
  }
}

}  // namespace wz
