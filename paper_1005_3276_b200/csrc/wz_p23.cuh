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

enum { P23_FFT = 0, P23_MULT = 1, P23_MULTPC = 2, P23_DIAGPC = 3, P23_MULTT = 4 };
// MULTT: MULT with c(p) read from the plan's table (args.ctab, one value per momentum site, built by k_ctab for the
// plan's rho) instead of one sqrt + one divide + one shuffle per site: the table (4 MB at 32^4 complex64) is shared by
// every source, spin component and launch and stays in the 126 MB L2.
// MULTPC: the multiply with args.pc = 1 or 2.  DIAGPC (two components per CTA only): the diagonal term of the same
// operator, accumulated onto the output of a MULTPC launch (there the CTA does not hold the other pair).
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
  const R* ctab;        // MULTT: c(p) = 2 rho / (s + Mw) per momentum site, [L0*L1][L3][L2] (n2 fastest)
};

// NC = spin components per CTA: 4 (whole plane quad, in place), or 2 when four planes
// do not fit in shared memory (64x64 complex128).  With NC = 2 the CTA with
// blockIdx.z = h reads components (2,3) [h = 0] or (0,1) [h = 1] and, for the multiply,
// writes the OTHER pair -- so in != out is required there (ping-pong buffers).
//
// Thread roles.  Role A (axis 2): per component slot, one line along x2 at fixed x3 per TPL2 lanes, lanes
// running along x3 (coalesced HBM accesses).  Role B (axis 3): per PAIR of component slots (the pairs the
// overlap multiply couples: (0,1) <-> (2,3)), every warp holds RPW = 16/TPL3 rows of BOTH components of the pair,
// component 0 of the pair in the low half of each group of G3 = 32/TPL3 lanes, component 1 in the high half.
// So the partner component of a momentum site sits in lane ^ RPW of the same warp and the multiply takes it by
// shuffle: the momentum-space exchange through shared memory (one store + two loads per element, two block
// barriers) of the first version of this kernel is gone, c(p) is shared between the two lanes by shuffle as well,
// and the results go back to the thread's own rows (the plane of input component c then holds output component c^2).
template <typename R, int L2, int L3, int T2, int T3, int NC = 4>
struct P23Cfg {
  static constexpr int TPL2 = T2, TPL3 = T3;  // lanes per line along axis 2 / axis 3
  static constexpr int NR2 = L2 / TPL2, NR3 = L3 / TPL3;
  static constexpr int NTC_A = (L3 * TPL2 + 31) / 32 * 32;  // threads per component slot in role A (whole warps)
  static constexpr int NT_A = NC * NTC_A;
  static constexpr int G3 = 32 / TPL3;          // line slots per warp in role B
  static constexpr int RPW = G3 / 2;            // rows per warp in role B (each row twice: both components of the pair)
  static constexpr int WPP = (L2 + RPW - 1) / RPW;  // warps per component pair
  static constexpr int NT_B = (NC / 2) * WPP * 32;
  static constexpr int NT = NT_A > NT_B ? NT_A : NT_B;
  static constexpr int PITCH = L3 + 1;            // row pitch (elements)
  // component pitch: the two half-groups of a role-B access (same rows, adjacent components) must fall into
  // different banks: complex64 (64-bit accesses, 16 lanes per wavefront): pitch = 8 mod 16 elements;
  // complex128 (128-bit accesses, 8 lanes per wavefront): pitch = 4 mod 8 elements
  static constexpr int CP_MOD = (sizeof(R) == 4) ? 16 : 8;
  static constexpr int CP_RAW = L2 * PITCH;
  static constexpr int CPITCH = CP_RAW + ((CP_MOD / 2 - CP_RAW % CP_MOD) + CP_MOD) % CP_MOD;
  static constexpr size_t SMEM = sizeof(cpx<R>) * NC * (size_t)CPITCH;
  static constexpr size_t SMEM_PC = SMEM;
  static_assert(NR3 % 2 == 0, "c(p) is shared between the two lanes of a pair, half of the line each");
};

template <typename R>
__device__ __forceinline__ R shfl_xor_r(R v, int dist) { return __shfl_xor_sync(0xffffffffu, v, dist); }

// Resident CTAs per SM the register allocation must allow (32x32 complex64 planes: the benchmark lattice).
// Measured at 32^4 x 12: 4 CTAs (no spills, 113 registers) 187 us per launch; 5 CTAs
// (12 bytes spilled) 198 us; 6 CTAs (260 bytes) 228 us.
template <typename R, int L2, int L3>
struct p23_minb {
  static constexpr int v = (sizeof(R) == 4 && L2 == 32 && L3 == 32) ? 4 : 1;
};

template <typename R, int L2, int L3, int T2, int T3, int MODE, int DIR, int NC = 4, typename S = cpx<R>>
__global__ void __launch_bounds__(P23Cfg<R, L2, L3, T2, T3, NC>::NT, p23_minb<R, L2, L3>::v)
k_p23(const P23Args<R> a) {
  using Cfg = P23Cfg<R, L2, L3, T2, T3, NC>;
  constexpr int TPL2 = Cfg::TPL2, TPL3 = Cfg::TPL3, NR2 = Cfg::NR2, NR3 = Cfg::NR3;
  constexpr int NTC_A = Cfg::NTC_A, PITCH = Cfg::PITCH, CPITCH = Cfg::CPITCH;
  constexpr int G3 = Cfg::G3, RPW = Cfg::RPW, WPP = Cfg::WPP;
  constexpr bool kDiag = (MODE == P23_DIAGPC);   // out += F^-1 (m or m^*)/D F in, component by component
  constexpr bool kPC = (MODE == P23_MULTPC);
  constexpr bool kTab = (MODE == P23_MULTT);     // c(p) from the table
  constexpr bool kMult = (MODE == P23_MULT || kPC || kTab);
  constexpr bool kMom = kMult || kDiag;          // works in momentum space between two transforms
  constexpr bool kStage = kPC && NC == 4;        // diagonal term of M0^-1 inside this launch (needs all four components)
  constexpr int D1 = kMom ? +1 : DIR;  // direction of the first half
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cpx<R>* sm = reinterpret_cast<cpx<R>*>(smem_raw);
  __shared__ R tb[kMom ? 2 * 4 * 64 : 1];

  const int bxr = a.rev ? (int)(gridDim.x - 1 - blockIdx.x) : (int)blockIdx.x;
  const int byr = a.rev ? (int)(gridDim.y - 1 - blockIdx.y) : (int)blockIdx.y;
  if (a.gate && !cg_active(a.gate + byr)) return;

  const int tid = threadIdx.x;
  const int plane = bxr;
  const long PL = (long)L2 * L3;
  const long fbase = (long)byr * 4 * a.nplanes;  // first field of this batch entry

  if constexpr (kMom) {
    for (int i = tid; i < 2 * 4 * 64; i += blockDim.x) tb[i] = a.tab[i];
  }

  // global spin component held by component slot s on input (cin) and on output (cout)
  const int half = (NC == 4) ? 0 : (int)blockIdx.z;
  auto cin_of = [&](int s) { return (NC == 4) ? s : (kMult ? (half ? s : 2 + s) : 2 * half + s); };
  auto cout_of = [&](int s) { return kMult ? (cin_of(s) ^ 2) : cin_of(s); };

  // role A: line along axis 2 at x3
  const int clA = tid / NTC_A;
  int x3A, jA;
  lane_split<TPL2>(tid % NTC_A, x3A, jA);
  const bool actA = (tid < Cfg::NT_A) && x3A < L3;
  cpx<R>* smA = sm + (actA ? clA : 0) * CPITCH;
  // role B: line along axis 3 at n2, both components of a pair in one warp
  const int wB = tid >> 5, lB = tid & 31;
  const int qB = lB % G3, jB = lB / G3;
  const int hB = qB / RPW;                               // component of the pair
  const int n2B = (wB % WPP) * RPW + (qB % RPW);
  const bool warpB = tid < Cfg::NT_B;                    // whole warps
  const bool actB = warpB && n2B < L2;
  const int slotB = warpB ? (wB / WPP) * 2 + hB : 0;
  cpx<R>* smB = sm + slotB * CPITCH + (actB ? n2B : 0) * PITCH;

  // Planes of the CTA one wave of resident CTAs further on -> L2 (one bulk prefetch per spin plane): that CTA then pays
  // L2 instead of HBM latency for its first loads.  Issued LATE (before the inverse axis-2 step, the last phase):
  // measured at 32^4 x 12 per launch: no prefetch 208 us; at CTA start, half a wave ahead 182; at CTA start, one wave
  // 183; after the axis-2 transform 183; before the inverse axis-2 step, half a wave 179, one wave 177, 1.5 waves 178.
  auto prefetch_planes = [&]() {
    if constexpr (NC == 4) {
      const int dist = a.pf_dist;
      if (dist > 0 && tid < 4) {
        const long lin = (long)blockIdx.y * gridDim.x + blockIdx.x + dist;
        if (lin < (long)gridDim.y * gridDim.x) {
          long by = lin / gridDim.x, bx = lin % gridDim.x;  // launch order -> data order
          if (a.rev) { by = gridDim.y - 1 - by; bx = gridDim.x - 1 - bx; }
          const S* pf = reinterpret_cast<const S*>(a.in) + ((by * 4 + tid) * a.nplanes + bx) * PL;
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(pf), "r"((unsigned)(PL * sizeof(S))));
        }
      }
    }
  };
  // ---- half 1, axis 2 (lanes run along x3: coalesced HBM reads) ----
  if (tid < Cfg::NT_A) {
    using F2 = LineFFT<R, L2, D1, VAR_DIT, TPL2>;
    const typename sptr<R, S>::type gin = as_stored<R, S>(a.in) + (fbase + (long)cin_of(clA) * a.nplanes + plane) * PL;
    cpx<R> x[NR2];
#pragma unroll
    for (int k = 0; k < NR2; ++k) {
      cpx<R> v = {R(0), R(0)};
      if (actA) v = gin[(long)F2::in_pos(k, jA) * L3 + x3A];
      x[k] = v;
    }
    F2::run(x, jA);
    if (actA) {
#pragma unroll
      for (int k = 0; k < NR2; ++k) smA[F2::out_pos(k, jA) * PITCH + x3A] = x[k];
    }
  }
  __syncthreads();

  // ---- axis 3: forward, [momentum-space multiply, inverse]; in registers, every row stays with its thread ----
  using F3 = LineFFT<R, L3, D1, VAR_DIT, TPL3>;
  using G3i = LineFFT<R, L3, -1, VAR_DIF, TPL3>;
  cpx<R> y[NR3];
  if (warpB) {
#pragma unroll
    for (int k = 0; k < NR3; ++k) {
      cpx<R> v = {R(0), R(0)};
      if (actB) v = smB[F3::in_pos(k, jB)];
      y[k] = v;
    }
    F3::run(y, jB);
    if constexpr (!kMom || kStage) {
      // plain transform: done.  M0^-1 with all four components here: the diagonal term needs the OTHER pair's
      // transformed rows, exchanged through shared memory
      if (actB) {
#pragma unroll
        for (int k = 0; k < NR3; ++k) smB[F3::out_pos(k, jB)] = y[k];
      }
    }
  }
  if constexpr (kStage) __syncthreads();
  if constexpr (kMom) {
    cpx<R> w[NR3];
    if (warpB) {
      const int n0 = plane / a.L1, n1 = plane % a.L1;
      const R* sn = tb;             // sin p_mu
      const R* sh = tb + 4 * 64;    // sin^2(p_mu/2)
      const int n2 = actB ? n2B : 0;
      const R s0 = sn[0 * 64 + n0], s1 = sn[1 * 64 + n1], s2 = sn[2 * 64 + n2];
      const R S012 = s0 * s0 + s1 * s1 + s2 * s2;
      const R Mw012 = a.rho - R(2) * (sh[0 * 64 + n0] + sh[1 * 64 + n1] + sh[2 * 64 + n2]);
      const R kk = R(2) * a.rho * a.sign * a.scale;  // 1/V of the inverse transform rides along
      const R m2 = a.m_re * a.m_re + a.m_im * a.m_im;
      // out_cc = i c(p) sign (Ca psi_a + Cb psi_b),  Ca = (A0, A1 + A3 s3), Cb = (B0, B1 + B3 s3), with (psi_a, psi_b)
      // the pair this warp holds; this thread forms the output component cc = (its own component) ^ 2
      const int cc = cout_of(slotB);
      R A0, A1, A3, B0, B1, B3;
      if (cc == 0)      { A0 = s0;  A1 = R(0); A3 = R(1);  B0 = s2;  B1 = s1;   B3 = R(0); }
      else if (cc == 1) { A0 = -s2; A1 = s1;   A3 = R(0);  B0 = s0;  B1 = R(0); B3 = R(-1); }
      else if (cc == 2) { A0 = s0;  A1 = R(0); A3 = R(-1); B0 = -s2; B1 = -s1;  B3 = R(0); }
      else              { A0 = s2;  A1 = -s1;  A3 = R(0);  B0 = s0;  B1 = R(0); B3 = R(1); }
      // this thread's own row is psi_a (hB = 0) or psi_b (hB = 1): coefficients of (own, partner)
      const R P0 = hB ? B0 : A0, P1 = hB ? B1 : A1, P3 = hB ? B3 : A3;
      const R Q0 = hB ? A0 : B0, Q1 = hB ? A1 : B1, Q3 = hB ? A3 : B3;
      // diagonal term of M0^-1 (pc = 1: upper components carry m, lower m^*) or of its conjugate transpose (pc = 2);
      // it multiplies psi_cc itself: the other pair's row (kStage), or this thread's own row (kDiag)
      const int cdiag = kDiag ? cin_of(slotB) : cc;
      const R dm_re = a.m_re;
      const R dm_im = ((cdiag < 2) == (a.pc == 1)) ? a.m_im : -a.m_im;
      [[maybe_unused]] const cpx<R>* smO = sm + (slotB ^ 2) * CPITCH + n2 * PITCH;  // kStage: same row, other pair
      if constexpr (kTab) {
        // c(p) from the table; sign and the 1/V of the inverse transform ride on the row coefficients
        const R ks = a.sign * a.scale;
        const R p0 = P0 * ks, p1 = P1 * ks, p3 = P3 * ks, q0 = Q0 * ks, q1 = Q1 * ks, q3 = Q3 * ks;
        // table layout [plane][n3][n2]: the 16 rows of a warp half read 16 consecutive values (one wavefront per load)
        const R* crow = a.ctab + (long)plane * L2 * L3 + n2;
        R cv[NR3];
#pragma unroll
        for (int k = 0; k < NR3; ++k) cv[k] = __ldg(crow + F3::out_pos(k, jB) * L2);
#pragma unroll
        for (int k = 0; k < NR3; ++k) {
          const int n3 = F3::out_pos(k, jB);
          const R s3 = sn[3 * 64 + n3];
          const cpx<R> own = y[k];
          const cpx<R> oth = shfl_xor_c(own, RPW);
          const R Pi = p1 + p3 * s3, Qi = q1 + q3 * s3;
          const R tr = p0 * own.re - Pi * own.im + q0 * oth.re - Qi * oth.im;
          const R ti = p0 * own.im + Pi * own.re + q0 * oth.im + Qi * oth.re;
          w[out_index<NR3>(k)] = {-cv[k] * ti, cv[k] * tr};  // times i c(p)
        }
      } else
#pragma unroll
      for (int k = 0; k < NR3 / 2; ++k) {
        // c(p) for registers k and k + NR3/2: this lane evaluates one, its pair partner (lane ^ RPW) the other
        const int n3lo = F3::out_pos(k, jB), n3hi = F3::out_pos(k + NR3 / 2, jB);
        const int n3m = hB ? n3hi : n3lo;
        const R s3m = sn[3 * 64 + n3m];
        const R S2m = S012 + s3m * s3m;
        R cfm = overlap_c(Mw012 - R(2) * sh[3 * 64 + n3m], S2m, kk);
        R dgm = R(0);
        if constexpr (kPC || kDiag) {  // cf carries rho-scaling and 1/V; c = cf / a.scale;  D = c^2 S2 + |m|^2
          const R c = cfm / a.scale;
          const R invD = R(1) / (c * c * S2m + m2);
          cfm *= invD;
          dgm = a.scale * invD;
        }
        const R cfo = shfl_xor_r(cfm, RPW);
        const R cf2[2] = {hB ? cfo : cfm, hB ? cfm : cfo};
        R dg2[2] = {R(0), R(0)};
        if constexpr (kPC || kDiag) {
          const R dgo = shfl_xor_r(dgm, RPW);
          dg2[0] = hB ? dgo : dgm;
          dg2[1] = hB ? dgm : dgo;
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int kr = k + e * (NR3 / 2);
          const int n3 = e ? n3hi : n3lo;
          const cpx<R> own = y[kr];
          cpx<R> o = {R(0), R(0)};
          if constexpr (kMult) {
            const R s3 = sn[3 * 64 + n3];
            const cpx<R> oth = shfl_xor_c(own, RPW);
            const R Pi = P1 + P3 * s3, Qi = Q1 + Q3 * s3;
            const R tr = P0 * own.re - Pi * own.im + Q0 * oth.re - Qi * oth.im;
            const R ti = P0 * own.im + Pi * own.re + Q0 * oth.im + Qi * oth.re;
            o = {-cf2[e] * ti, cf2[e] * tr};  // times i
          }
          if constexpr (kStage || kDiag) {  // + (m or m^*) / D psi_cc
            cpx<R> d = own;
            if constexpr (kStage) d = smO[n3];
            const R dr = dm_re * dg2[e], di = dm_im * dg2[e];
            o.re += dr * d.re - di * d.im;
            o.im += dr * d.im + di * d.re;
          }
          w[out_index<NR3>(kr)] = o;
        }
      }
    }
    if constexpr (kStage) __syncthreads();  // every read of the staged rows is done
    if (warpB) {
      G3i::run(w, jB);
      if (actB) {
#pragma unroll
        for (int k = 0; k < NR3; ++k) smB[G3i::out_pos(k, jB)] = w[k];
      }
    }
  }
  __syncthreads();

  if constexpr (MODE == P23_FFT) {
    // coalesced copy-out of the planes
    for (int i = tid; i < NC * L2 * L3; i += blockDim.x) {
      const int ci = i / (L2 * L3), r = i % (L2 * L3);
      const int n2 = r / L3, n3 = r % L3;
      cpx<R> v = sm[ci * CPITCH + n2 * PITCH + n3];
      as_stored<R, S>(a.out)[(fbase + (long)cout_of(ci) * a.nplanes + plane) * PL + r] = cscale(v, a.scale);
    }
  } else {
    prefetch_planes();
    // ---- inverse axis 2, coalesced HBM writes; slot s now holds output component cout_of(s) ----
    if (tid < Cfg::NT_A) {
      using G2 = LineFFT<R, L2, -1, VAR_DIT, TPL2>;
      const typename sptr<R, S>::type gout = as_stored<R, S>(a.out) + (fbase + (long)cout_of(clA) * a.nplanes + plane) * PL;
      cpx<R> x[NR2];
#pragma unroll
      for (int k = 0; k < NR2; ++k) {
        cpx<R> v = {R(0), R(0)};
        if (actA) v = smA[G2::in_pos(k, jA) * PITCH + x3A];
        x[k] = v;
      }
      G2::run(x, jA);
      if (actA) {
#pragma unroll
        for (int k = 0; k < NR2; ++k) {
          const long di = (long)G2::out_pos(k, jA) * L3 + x3A;
          if constexpr (kDiag) {  // accumulate onto what the off-diagonal launch wrote
            const cpx<R> prev = gout[di];
            x[k] = {x[k].re + prev.re, x[k].im + prev.im};
          }
          gout[di] = x[k];
        }
      }
    }
  }
}

// c(p) = 2 rho / (s + Mw) (cancellation-free branch for Mw < 0) at every momentum site, for P23_MULTT.
template <typename R>
__global__ void k_ctab(R* __restrict__ ctab, const R* __restrict__ tab, int L0, int L1, int L2, int L3, R rho) {
  const long V = (long)L0 * L1 * L2 * L3;
  const R* sn = tab;
  const R* sh = tab + 4 * 64;
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long)gridDim.x * blockDim.x) {
    long t = i;
    const int n3 = (int)(t % L3); t /= L3;
    const int n2 = (int)(t % L2); t /= L2;
    const int n1 = (int)(t % L1); t /= L1;
    const int n0 = (int)t;
    const R s0 = sn[0 * 64 + n0], s1 = sn[1 * 64 + n1], s2 = sn[2 * 64 + n2], s3 = sn[3 * 64 + n3];
    const R S2 = s0 * s0 + s1 * s1 + s2 * s2 + s3 * s3;
    const R Mw = rho - R(2) * (sh[0 * 64 + n0] + sh[1 * 64 + n1] + sh[2 * 64 + n2] + sh[3 * 64 + n3]);
    ctab[(((long)n0 * L1 + n1) * L3 + n3) * L2 + n2] = overlap_c(Mw, S2, R(2) * rho);  // [plane][n3][n2]
  }
}

}  // namespace wz
