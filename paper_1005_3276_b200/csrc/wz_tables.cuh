// wz_tables.cuh -- host-side kernel dispatch tables: which instantiation of k_p01 / k_p23 serves
// which lattice, with its launch shape, and the tuning choices (lanes per line, tile width).
// The kernels are instantiated in wz_kmod.cu, compiled once per module (-DWZ_MOD=n) so that the
// modules build in parallel; wz_lib.cu gathers their entries.
#pragma once
#include <vector>

#include "wz_p01.cuh"
#include "wz_p23.cuh"

namespace wz {

// One (x0,x1)-pass kernel with its launch shape.
template <typename R>
struct P01Kern {
  void (*fn)(const P01Args<R>) = nullptr;
  int nt = 0, nseg = 0;
  int l0 = 0, l1 = 0;   // tile extents along axes 0, 1 (for the TMA tile prefetch)
  int half = 0;         // 1: binary16 storage of t, chi, r, p (cpxh)
  int fin = FIN_STORE;  // what k_finalize does with the kernel's reduction (if it has one)
  bool split_finalize = false;  // the kernel leaves partials; k_finalize<fin> must follow (p01_split_finalize)
  size_t smem = 0;
};
template <typename R>
struct P01Entry {
  int L0, L1;
  long I;  // (x2,x3) volume the kernels were specialised for; 0 = any (run-time)
  int half = 0;  // 1: t, chi, r, p are stored as cpxh (two binary16 values per complex number); only the CG-fused modes are set
  P01Kern<R> fwd, inv, mid, mid_pq, end, fwdcg, endcg;
  P01Kern<R> fwdcg_s, endcg_s;  // shifted system (M^dag M + sigma): A' also reduces <p,p>, E' adds sigma p to q
  int nseg() const {  // largest tile width of the entry: the (x2,x3) volume must be a multiple
    int m = 1;
    for (const P01Kern<R>* k : {&fwd, &inv, &mid, &mid_pq, &end, &fwdcg, &endcg, &fwdcg_s, &endcg_s}) if (k->fn) m = k->nseg > m ? k->nseg : m;
    return m;
  }
  int min_nseg() const {
    int m = 1 << 30;
    for (const P01Kern<R>* k : {&fwd, &inv, &mid, &mid_pq, &end, &fwdcg, &endcg, &fwdcg_s, &endcg_s}) if (k->fn) m = k->nseg < m ? k->nseg : m;
    return m;
  }
};
template <typename R>
struct P23Entry {
  int half = 0;  // 1: binary16 storage (cpxh); only `mult` / `multt` are set
  int L2, L3, nt, nhalf;  // nhalf = 2: two components per CTA, grid.z = 2, multiply needs in != out
  size_t smem, smem_pc;
  void (*fwd)(const P23Args<R>);
  void (*inv)(const P23Args<R>);
  void (*mult)(const P23Args<R>);
  void (*multpc)(const P23Args<R>);  // multiply with the free inverse (preconditioner)
  void (*multt)(const P23Args<R>) = nullptr;   // multiply with c(p) from the plan's table (P23_MULTT)
  void (*diagpc)(const P23Args<R>) = nullptr;  // nhalf = 2 only: diagonal term of the free inverse, accumulated (wz_p23.cuh)
};

// ---- tuning: lanes per lattice line (TPL) and tile width (NSEG) -------------------
// More lanes per line = fewer registers per thread and more resident warps; one radix-2 shuffle
// step per doubling.  32-long complex64 lines are held whole by one thread in every mode
// (TPL = 1: no shuffle steps, 24-35 % fewer instructions, 32 independent loads in flight; pass A'
// 441 -> 427 us, pass E' 330 -> 317 us per launch at 32^4 x 12); 48- and 64-long lines take two lanes.
template <typename R, int L, int MODE> struct tune_tpl {   // axes 0,1
  static constexpr int v = (sizeof(R) == 4) ? (L >= 48 ? 2 : 1) : (L >= 48 ? 4 : (L >= 24 ? 2 : 1));
};
template <typename R, int L> struct tune_tpl23 {  // axes 2,3
  static constexpr int v = (sizeof(R) == 4) ? (L >= 48 ? 2 : 1) : (L >= 48 ? 4 : (L >= 24 ? 2 : 1));
};
// NSEG: consecutive (x2,x3) sites per strided tile: tile L0 x L1 x NSEG <= 136 KB.  Each (x0,x1) row
// contributes one run of NSEG*8 bytes, and every run costs one L1 tag lookup per access: at 32^4
// complex64 going from 32-byte to 64-/128-byte runs took the iteration from 173 to 141 us per source.
// Inverse modes and pass A': 128-byte runs, one 512-thread CTA per SM; the stand-alone forward mode: 64-byte runs, two
// 256-thread CTAs per SM.  (Pass A' with 128-byte runs lost before it had the TMA tile prefetch, 457 against 434 us; with
// it A' is unchanged, 437 against 435 us, and the passes around it run 1-2 % faster: 8307 -> 8380 it/s on the same box.)
template <typename R, int L0, int L1, int MODE> struct tune_nseg {
  static constexpr bool fwd = (MODE == P01_FWD || MODE == P01_FWDCG);
  static constexpr int v = (L1 == 1) ? (int)(512 / (2 * sizeof(R)))  // single-axis pass: 512-byte runs, no tile in shared memory
                         : (sizeof(R) == 4) ? (L0 * L1 > 2048 ? 4 : (L0 * L1 == 1024 ? (MODE == P01_FWD ? 8 : 16) : 8))
                                            : (L0 * L1 > 2048 ? 2 : 4);
};

template <typename R, int L0, int L1, int MODE, int FIN, int IC>
P01Kern<R> make_p01_kern() {
  constexpr int NSEG = tune_nseg<R, L0, L1, MODE>::v, T0 = tune_tpl<R, L0, MODE>::v, T1 = tune_tpl<R, L1, MODE>::v;
  using C = P01Cfg<R, L0, L1, NSEG, T0, T1>;
  P01Kern<R> k;
  k.fn = k_p01<R, L0, L1, NSEG, T0, T1, MODE, FIN, IC>;
  k.nt = C::NT; k.nseg = NSEG; k.smem = C::SMEM; k.l0 = L0; k.l1 = L1; k.fin = FIN; k.split_finalize = p01_split_finalize<L0, L1>::v;
  return k;
}
template <typename R, int L0, int L1, int IC = 0>
P01Entry<R> make_p01() {
  P01Entry<R> e;
  e.L0 = L0; e.L1 = L1; e.I = IC;
  e.fwd = make_p01_kern<R, L0, L1, P01_FWD, FIN_STORE, IC>();
  e.inv = make_p01_kern<R, L0, L1, P01_INV, FIN_STORE, IC>();
  e.mid = make_p01_kern<R, L0, L1, P01_MID, FIN_STORE, IC>();
  e.mid_pq = make_p01_kern<R, L0, L1, P01_MID, FIN_PQ, IC>();
  e.end = make_p01_kern<R, L0, L1, P01_END, FIN_STORE, IC>();
  e.fwdcg = make_p01_kern<R, L0, L1, P01_FWDCG, FIN_STORE, IC>();
  e.endcg = make_p01_kern<R, L0, L1, P01_ENDCG, FIN_RR, IC>();
  e.fwdcg_s = make_p01_kern<R, L0, L1, P01_FWDCG, FIN_PP, IC>();
  e.endcg_s = make_p01_kern<R, L0, L1, P01_ENDCG, FIN_RRS, IC>();
  return e;
}
template <typename R, int L2, int L3, int NC = 4>
P23Entry<R> make_p23() {
  constexpr int T2 = tune_tpl23<R, L2>::v, T3 = tune_tpl23<R, L3>::v;
  using C = P23Cfg<R, L2, L3, T2, T3, NC>;
  P23Entry<R> e;
  e.L2 = L2; e.L3 = L3; e.nt = C::NT; e.smem = C::SMEM; e.smem_pc = C::SMEM_PC; e.nhalf = 4 / NC;
  e.fwd = k_p23<R, L2, L3, T2, T3, P23_FFT, +1, NC>;
  e.inv = k_p23<R, L2, L3, T2, T3, P23_FFT, -1, NC>;
  e.mult = k_p23<R, L2, L3, T2, T3, P23_MULT, +1, NC>;
  e.multpc = k_p23<R, L2, L3, T2, T3, P23_MULTPC, +1, NC>;
  e.multt = k_p23<R, L2, L3, T2, T3, P23_MULTT, +1, NC>;
  if constexpr (NC == 2) e.diagpc = k_p23<R, L2, L3, T2, T3, P23_DIAGPC, +1, NC>;
  return e;
}

// ---- binary16 storage (NEXT-3): the three CG-fused (x0,x1) passes and the multiply pass with S = cpxh.
// Tiles of 16 sites in every mode at 32x32 (64-byte runs of 4-byte elements; the shared-memory tile stays complex64).
template <int L0, int L1, int MODE> struct tune_nseg_half {
  static constexpr int v = (L0 * L1 == 1024) ? 16 : 8;
};
template <int L0, int L1, int MODE, int FIN, int IC>
P01Kern<float> make_p01_kern_half() {
  using R = float;
  constexpr int NSEG = tune_nseg_half<L0, L1, MODE>::v, T0 = tune_tpl<R, L0, MODE>::v, T1 = tune_tpl<R, L1, MODE>::v;
  using C = P01Cfg<R, L0, L1, NSEG, T0, T1>;
  P01Kern<R> k;
  k.fn = k_p01<R, L0, L1, NSEG, T0, T1, MODE, FIN, IC, cpxh>;
  k.half = 1;
  k.nt = C::NT; k.nseg = NSEG; k.smem = C::SMEM; k.l0 = L0; k.l1 = L1; k.fin = FIN; k.split_finalize = p01_split_finalize<L0, L1>::v;
  return k;
}
template <int L0, int L1, int IC = 0>
P01Entry<float> make_p01_half() {
  P01Entry<float> e;
  e.L0 = L0; e.L1 = L1; e.I = IC; e.half = 1;
  e.fwdcg = make_p01_kern_half<L0, L1, P01_FWDCG, FIN_STORE, IC>();
  e.mid_pq = make_p01_kern_half<L0, L1, P01_MID, FIN_PQ, IC>();
  e.endcg = make_p01_kern_half<L0, L1, P01_ENDCG, FIN_RR, IC>();
  return e;
}
template <int L2, int L3>
P23Entry<float> make_p23_half() {
  using R = float;
  constexpr int T2 = tune_tpl23<R, L2>::v, T3 = tune_tpl23<R, L3>::v;
  using C = P23Cfg<R, L2, L3, T2, T3, 4>;
  P23Entry<R> e;
  e.half = 1;
  e.L2 = L2; e.L3 = L3; e.nt = C::NT; e.smem = C::SMEM; e.smem_pc = C::SMEM_PC; e.nhalf = 1;
  e.fwd = nullptr; e.inv = nullptr; e.multpc = nullptr;
  e.mult = k_p23<R, L2, L3, T2, T3, P23_MULT, +1, 4, cpxh>;
  e.multt = k_p23<R, L2, L3, T2, T3, P23_MULTT, +1, 4, cpxh>;
  return e;
}

// One kernel module = one translation unit of wz_kmod.cu.  The twiddle tables are __constant__
// memory, private to each translation unit (and per device): every module uploads its own copy.
struct KernelModule {
  bool (*upload_twiddles)(const void* tf /* float2[TWN] */, const void* td /* double2[TWN] */);
  void (*p01f)(std::vector<P01Entry<float>>&);
  void (*p01d)(std::vector<P01Entry<double>>&);
  void (*p23f)(std::vector<P23Entry<float>>&);
  void (*p23d)(std::vector<P23Entry<double>>&);
};
constexpr int kNumKernelModules = 8;
const KernelModule* kernel_module(int i);  // wz_lib.cu
#define WZ_DECLARE_MODULE(n) const KernelModule* wz_kernel_module_##n();
WZ_DECLARE_MODULE(0) WZ_DECLARE_MODULE(1) WZ_DECLARE_MODULE(2) WZ_DECLARE_MODULE(3)
WZ_DECLARE_MODULE(4) WZ_DECLARE_MODULE(5) WZ_DECLARE_MODULE(6) WZ_DECLARE_MODULE(7)
#undef WZ_DECLARE_MODULE

}  // namespace wz
