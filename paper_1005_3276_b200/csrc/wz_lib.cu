// wz_lib.cu -- host side of the C-ABI in include/wz.h: plans, tables, kernel
// dispatch, the matvec pass schedule and the CG driver.  sm_100a only; there is no
// CPU path: every entry point either enqueues kernels or returns an error.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <map>
#include <mutex>
#include <set>
#include <vector>

#include <cuda.h>  // CUtensorMap types only; cuTensorMapEncodeTiled is resolved at run time (no libcuda link)

#include "../../include/wz.h"
#include "wz_cgk.cuh"
#include "wz_tables.cuh"

using namespace wz;

namespace wz {
const KernelModule* kernel_module(int i) {
  switch (i) {
    case 0: return wz_kernel_module_0();
    case 1: return wz_kernel_module_1();
    case 2: return wz_kernel_module_2();
    case 3: return wz_kernel_module_3();
    case 4: return wz_kernel_module_4();
    case 5: return wz_kernel_module_5();
    case 6: return wz_kernel_module_6();
    default: return wz_kernel_module_7();
  }
}
}  // namespace wz

namespace {

thread_local char g_err[512] = "";

bool cuda_ok(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
  return false;
}
#define WZ_CUDA(call)                                   \
  do {                                                  \
    if (!cuda_ok((call), #call)) return WZ_ECUDA;       \
  } while (0)

// ---- kernel dispatch tables: gathered from the kernel modules (wz_kmod.cu) ----------
template <typename R> struct tables;
template <> struct tables<float> {
  static void gather(std::vector<P01Entry<float>>& a, std::vector<P23Entry<float>>& b) {
    for (int i = 0; i < kNumKernelModules; ++i) { kernel_module(i)->p01f(a); kernel_module(i)->p23f(b); }
  }
};
template <> struct tables<double> {
  static void gather(std::vector<P01Entry<double>>& a, std::vector<P23Entry<double>>& b) {
    for (int i = 0; i < kNumKernelModules; ++i) { kernel_module(i)->p01d(a); kernel_module(i)->p23d(b); }
  }
};
template <typename R>
const std::vector<P01Entry<R>>& p01_table() {
  static const std::vector<P01Entry<R>> t = [] {
    std::vector<P01Entry<R>> a; std::vector<P23Entry<R>> b;
    tables<R>::gather(a, b);
    // entries specialised for one (x2,x3) volume come first (find_p01 takes the first match)
    std::stable_sort(a.begin(), a.end(), [](const P01Entry<R>& x, const P01Entry<R>& y) { return (x.I != 0) > (y.I != 0); });
    return a;
  }();
  return t;
}
template <typename R>
const std::vector<P23Entry<R>>& p23_table() {
  static const std::vector<P23Entry<R>> t = [] {
    std::vector<P01Entry<R>> a; std::vector<P23Entry<R>> b;
    tables<R>::gather(a, b);
    return b;
  }();
  return t;
}
template <typename R>
const P01Entry<R>* find_p01(int L0, int L1, long I, int half = 0) {
  for (const auto& e : p01_table<R>())  // specialised entries come first
    if (e.half == half && e.L0 == L0 && e.L1 == L1 && (e.I == 0 || e.I == I)) return &e;
  return nullptr;
}
template <typename R>
const P23Entry<R>* find_p23(int L2, int L3, int half = 0) {
  for (const auto& e : p23_table<R>())
    if (e.half == half && e.L2 == L2 && e.L3 == L3) return &e;
  return nullptr;
}

template <typename K>
bool set_smem(K kernel, size_t bytes);
template <typename R>
bool set_smem_kern(const P01Kern<R>& k) {
  return set_smem(k.fn, k.smem);
}
template <typename K>
bool set_smem(K kernel, size_t bytes) {
  if (bytes <= 32 * 1024) return true;  // static shared memory (tables, reduction scratch) counts against the 48 KB default too
  return cuda_ok(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes),
                 "cudaFuncSetAttribute(MaxDynamicSharedMemorySize)");
}

// ---- per-precision operator workspace -------------------------------------------
template <typename R>
struct OpWS {
  const P01Entry<R>* p01 = nullptr;
  const P23Entry<R>* p23 = nullptr;
  // single-axis decomposition of the (x0,x1) pass (64x64 lattices: a two-axis tile with runs longer than 32 bytes does
  // not fit in shared memory): p0s transforms axis 0 (all modes; inner volume L1*I), p1s axis 1 (x0 slices as fields)
  const P01Entry<R>* p0s = nullptr;
  const P01Entry<R>* p1s = nullptr;
  R* tab = nullptr;        // momentum tables [2][4][64]
  R* ctab = nullptr;       // c(p) per momentum site for the rho below (ensure_ctab); V entries
  R ctab_rho = R(-1);
  cpx<R>* t = nullptr;     // FFT temporary, max_batch spinors
  cpx<R>* t2 = nullptr;    // second FFT temporary (only where the multiply pass is out of place)
  cpx<R>* chi = nullptr;   // chi = M psi,   max_batch spinors
};

}  // namespace

// Everything the kernels of one CG iteration are launched with (the captured graph is valid for exactly these).
struct IterGraphKey {
  const void *phi, *r, *p, *x;
  double m[2], g[2], rho, sigma;
  int nb, pc, prec, block;
};

struct wz_plan {
  int L[4];
  long V, I;
  wz_dtype dtype;
  int max_batch;
  cudaStream_t stream;
  cudaStream_t lstream;    // where kernels are enqueued: `stream`, or `cap_stream` while a graph is being captured
  unsigned long long bytes = 0, launches = 0;
  double rho_tab = -1.0;  // rho the momentum tables do not depend on; kept for clarity
  OpWS<float> wsf;
  OpWS<double> wsd;        // always present: complex128 operator (plans of both dtypes)
  // CG vectors
  void *r = nullptr, *p = nullptr, *xs = nullptr;  // plan dtype, max_batch spinors each
  cpx<double>* q128 = nullptr;    // A X in complex128 (reliable updates, true residual), one spinor
  cpx<double>* phi128 = nullptr;  // C64 plans: phi widened
  cpx<double>* btilde128 = nullptr;  // C64 plans, preconditioned solves: (M0^-1)^dag b in complex128, per source
  cpx<double>* ratX = nullptr;       // wz_rational_apply: the X_i of the current shift(s), ratX_cap spinors
  size_t ratX_cap = 0;
  // multi-shift CG: search directions and (complex64 plans) solutions of every shift, [shift][source] spinors
  void *ms_p = nullptr, *ms_x = nullptr;
  size_t ms_cap = 0;               // spinors each of ms_p / ms_x holds
  MSState* ms_state = nullptr;     // [max_batch]
  double* ms_true = nullptr;       // [WZ_MAX_SHIFTS][max_batch] true residual norms squared
  OpWS<float> wsh;                 // binary16-storage operator workspace (wz_cg_solve_dc_half): t, chi hold cpxh
  void *h_r = nullptr, *h_p = nullptr;  // its r, p (cpxh), max_batch spinors each
  void* ms_rhs = nullptr;          // complex64 plans: defect of one shift, max_batch spinors (plan dtype)
  cpx<double>* ms_e = nullptr;     // complex64 plans: correction of the polishing solve, max_batch spinors
  double* partials = nullptr;
  unsigned* counter = nullptr;
  CGState* d_state = nullptr;
  CGState* h_state = nullptr;  // pinned, 2 slots
  cudaEvent_t ev[2] = {nullptr, nullptr};
  int npartials = 0;
  int num_sms = 148;
  int sweep = 0;  // direction of the last pass launched (next_sweep)
  int dev = 0;    // CUDA device the plan lives on; every entry point switches to it
  std::map<const void*, int> occ_cache;  // resident CTAs per wave, per kernel (wave_ctas)
  std::vector<void*> allocs;
  // optional per-kernel timing (wz_plan_profile): event pairs around sampled launches
  int profile = 0;
  int prof_override = -1;  // >= 0: record launches under this kind (reliable-update matvecs -> other)
  std::vector<cudaEvent_t> prof_ev;      // 2 per recorded launch
  std::vector<int> prof_kind;
  double prof_ms[WZ_NKINDS] = {0};
  unsigned long long prof_n[WZ_NKINDS] = {0};
  // CUDA graph of one chunk of CG iterations (north star iii): captured once per distinct set of
  // solve arguments on a private stream, replayed on `stream`
  int use_graph = 1;
  int tile_prefetch = 1;  // wave-ahead TMA prefetch of the strided input tiles of passes C and A'
  int no_ctab = 0;  // 1: never build the c(p) table (wz_apply_MdagM_noalloc: no device allocation)
  int block = 0;  // sources per block of the CG iteration (0: the whole batch in lock step)
  cudaStream_t cap_stream = nullptr;
  cudaGraphExec_t iter_graph = nullptr;
  IterGraphKey iter_key;
  int iter_graph_launches = 0;
  // residual history of the last solve as the host saw it at its convergence checks: per source (iteration, ||r||/||b||)
  std::vector<std::vector<std::pair<int, double>>> hist;
};

namespace {

const double kPi = 3.14159265358979323846264338327950288;

// Switches to the plan's device for the duration of an entry point and back.
struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) { ok = false; return; }
    if (cur != dev) {
      ok = cudaSetDevice(dev) == cudaSuccess;
      if (ok) prev = cur;
    }
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define WZ_ON_DEVICE(pl)                                                        \
  DeviceGuard wz_dev_guard((pl)->dev);                                          \
  if (!wz_dev_guard.ok) { snprintf(g_err, sizeof(g_err), "cudaSetDevice(%d) failed", (pl)->dev); return WZ_ECUDA; }

// exp(-2 pi i j/TWN) in both precisions.  __constant__ memory is per device: written once per
// device of the process (the current one), under a lock.
bool init_twiddles(int dev) {
  static std::mutex mu;
  static std::set<int> done;
  std::lock_guard<std::mutex> lock(mu);
  if (done.count(dev)) return true;
  std::vector<float2> tf(TWN);
  std::vector<double2> td(TWN);
  for (int j = 0; j < TWN; ++j) {
    // exact values on the axes and diagonals, symmetric elsewhere (octant reduction)
    int o = j % TWN;
    double ang = 2.0 * kPi * (double)o / (double)TWN;
    double c = std::cos(ang), s = std::sin(ang);
    if (o % (TWN / 4) == 0) {
      const int qd = o / (TWN / 4);
      c = (qd == 0) ? 1.0 : (qd == 2) ? -1.0 : 0.0;
      s = (qd == 1) ? 1.0 : (qd == 3) ? -1.0 : 0.0;
    }
    td[j] = make_double2(c, -s);
    tf[j] = make_float2((float)c, (float)-s);
  }
  for (int i = 0; i < kNumKernelModules; ++i)
    if (!kernel_module(i)->upload_twiddles(tf.data(), td.data()))
      return cuda_ok(cudaGetLastError(), "cudaMemcpyToSymbol(twiddles)") && false;
  done.insert(dev);
  return true;
}

template <typename T>
bool dev_alloc(wz_plan* pl, T** ptr, size_t count) {
  void* p = nullptr;
  size_t bytes = count * sizeof(T);
  if (bytes == 0) bytes = sizeof(T);
  cudaError_t e = cudaMalloc(&p, bytes);
  if (e != cudaSuccess) {
    snprintf(g_err, sizeof(g_err), "cudaMalloc(%zu bytes): %s", bytes, cudaGetErrorString(e));
    cudaGetLastError();
    return false;
  }
  pl->allocs.push_back(p);
  pl->bytes += bytes;
  *ptr = reinterpret_cast<T*>(p);
  return true;
}

// Momentum tables (p0 = 2 pi (n0 + 1/2)/T, p_i = 2 pi n_i/L_i),
// computed in double on the host: tab[0][mu][n] = sin p_mu, tab[1][mu][n] = sin^2(p_mu/2).
int wave_ctas(wz_plan* pl, const void* fn, int nt, size_t smem);

template <typename R>
wz_status setup_ws(wz_plan* pl, OpWS<R>& ws, int nbatch_t) {
  ws.p01 = find_p01<R>(pl->L[0], pl->L[1], pl->I);
  ws.p23 = find_p23<R>(pl->L[2], pl->L[3]);
  if (!ws.p01 || !ws.p23) return WZ_EUNSUPPORTED;
  if (pl->I % ws.p01->nseg()) return WZ_EUNSUPPORTED;
  if (pl->L[0] * pl->L[1] > 2048) {
    const auto* e0 = find_p01<R>(pl->L[0], 1, 0);
    const auto* e1 = find_p01<R>(pl->L[1], 1, 0);
    if (e0 && e1 && ((long)pl->L[1] * pl->I) % e0->nseg() == 0 && pl->I % e1->nseg() == 0) { ws.p0s = e0; ws.p1s = e1; }
  }
  const P01Entry<R>* entries[3] = {ws.p01, ws.p0s, ws.p1s};
  for (const P01Entry<R>* a : entries) {
    if (!a) continue;
    if (!set_smem_kern(a->fwdcg_s) || !set_smem_kern(a->endcg_s)) return WZ_ECUDA;
    if (!set_smem_kern(a->fwd) || !set_smem_kern(a->inv) || !set_smem_kern(a->mid) ||
        !set_smem_kern(a->mid_pq) || !set_smem_kern(a->end) || !set_smem_kern(a->fwdcg) ||
        !set_smem_kern(a->endcg))
      return WZ_ECUDA;
  }
  const auto* b = ws.p23;
  if (!set_smem(b->fwd, b->smem) || !set_smem(b->inv, b->smem) || !set_smem(b->mult, b->smem) ||
      !set_smem(b->multpc, b->smem_pc) || (b->diagpc && !set_smem(b->diagpc, b->smem_pc)) ||
      (b->multt && !set_smem(b->multt, b->smem)))
    return WZ_ECUDA;
  wave_ctas(pl, (const void*)b->mult, b->nt, b->smem);  // occupancy queries now, not inside a stream capture
  wave_ctas(pl, (const void*)b->multpc, b->nt, b->smem_pc);
  if (b->multt) wave_ctas(pl, (const void*)b->multt, b->nt, b->smem);
  if (b->diagpc) wave_ctas(pl, (const void*)b->diagpc, b->nt, b->smem_pc);
  wave_ctas(pl, (const void*)b->fwd, b->nt, b->smem);
  wave_ctas(pl, (const void*)b->inv, b->nt, b->smem);
  std::vector<R> h(2 * 4 * 64, R(0));
  for (int mu = 0; mu < 4; ++mu)
    for (int n = 0; n < pl->L[mu]; ++n) {
      const double p = 2.0 * kPi * ((double)n + (mu == 0 ? 0.5 : 0.0)) / (double)pl->L[mu];
      const double sh = std::sin(0.5 * p);
      h[(0 * 4 + mu) * 64 + n] = (R)std::sin(p);
      h[(1 * 4 + mu) * 64 + n] = (R)(sh * sh);
    }
  if (!dev_alloc(pl, &ws.tab, h.size())) return WZ_ENOMEM;
  WZ_CUDA(cudaMemcpyAsync(ws.tab, h.data(), sizeof(R) * h.size(), cudaMemcpyHostToDevice, pl->stream));
  WZ_CUDA(cudaStreamSynchronize(pl->stream));
  const size_t n = (size_t)nbatch_t * 4 * pl->V;
  if (!dev_alloc(pl, &ws.t, n) || !dev_alloc(pl, &ws.chi, n)) return WZ_ENOMEM;
  if (ws.p23->nhalf == 2 && !dev_alloc(pl, &ws.t2, n)) return WZ_ENOMEM;
  return WZ_OK;
}

constexpr size_t kProfMaxPairs = 8192;
// Bracket the next launch with events when profiling (bounded number of samples).
struct ProfScope {
  wz_plan* pl; int kind; bool on = false;
  ProfScope(wz_plan* p, int k) : pl(p), kind(p->prof_override >= 0 ? p->prof_override : k) {
    if (pl->profile && pl->prof_kind.size() < kProfMaxPairs) {
      cudaEvent_t a, b;
      if (cudaEventCreate(&a) == cudaSuccess && cudaEventCreate(&b) == cudaSuccess) {
        cudaEventRecord(a, pl->lstream);
        pl->prof_ev.push_back(a); pl->prof_ev.push_back(b); pl->prof_kind.push_back(kind);
        on = true;
      }
    }
  }
  ~ProfScope() { if (on) cudaEventRecord(pl->prof_ev.back(), pl->lstream); pl->launches++; }
};

template <typename R, typename A>
wz_status launch(wz_plan* pl, int kind, void (*k)(const A), dim3 grid, int nt, size_t smem, const A& args) {
  {
    ProfScope ps(pl, kind);
    k<<<grid, nt, smem, pl->lstream>>>(args);
  }
  WZ_CUDA(cudaGetLastError());
  return WZ_OK;
}

// Wave-ahead L2 prefetch of the contiguous pass (wz_p23.cuh): distance = the CTAs resident on the whole GPU at once
// (one wave), issued late in the CTA (measurements there).
constexpr int kPrefetchPercent = 100;
int wave_ctas(wz_plan* pl, const void* fn, int nt, size_t smem) {
  auto it = pl->occ_cache.find(fn);
  if (it != pl->occ_cache.end()) return it->second;
  int occ = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, nt, smem) != cudaSuccess || occ < 1) occ = 1;
  return pl->occ_cache[fn] = occ * pl->num_sms;
}

// Alternating sweep direction: consecutive passes run over the tiles in opposite orders, so the first CTAs
// of a launch read what the previous launch wrote (or read) last and the 126 MB L2 still holds.  Every CTA's
// work and every reduction slot is indexed by the tile, not by blockIdx, so results do not depend on it.
int next_sweep(wz_plan* pl) {
  pl->sweep ^= 1;
  return pl->sweep;
}

// ---- TMA descriptor of a field array [nf][l0][l1][inner] of complex<R>, box = one strided tile l0 x l1 x nseg ----
// Rank 4 in reals: (2*inner, l1, l0, nf), box (2*nseg, l1, l0, 1).  Host-side encoding only (no device work, no
// allocation); used by k_p01 to prefetch whole tiles into L2 (wz_p01.cuh).  Returns false where the driver entry
// point is missing or the shape is outside the TMA limits: the kernels then run without the prefetch.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    cudaGetLastError();
    return (EncodeTiledFn)p;
  }();
  return fn;
}
template <typename R>
bool make_tile_tmap(TMapBlob* out, const void* base, long inner, int l0, int l1, int nseg, long nf, bool half = false) {
  const size_t esz = half ? 2 : sizeof(R);  // bytes of one real number as stored
  static_assert(sizeof(CUtensorMap) == sizeof(TMapBlob), "CUtensorMap is 128 bytes");
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc || !base || ((uintptr_t)base & 15) || l0 > 256 || l1 > 256 || 2 * nseg > 256) return false;
  if ((2 * nseg * esz) % 16 || (inner * 2 * esz) % 16) return false;
  const cuuint64_t gdim[4] = {(cuuint64_t)(2 * inner), (cuuint64_t)l1, (cuuint64_t)l0, (cuuint64_t)nf};
  const cuuint64_t gstr[3] = {(cuuint64_t)(2 * inner * esz), (cuuint64_t)(2 * inner * esz) * l1,
                              (cuuint64_t)(2 * inner * esz) * l1 * l0};
  const cuuint32_t box[4] = {(cuuint32_t)(2 * nseg), (cuuint32_t)l1, (cuuint32_t)l0, 1u};
  const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
  CUtensorMap tm;
  const CUresult r = enc(&tm, half ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : (sizeof(R) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64), 4u,
                         const_cast<void*>(base), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  memcpy(out, &tm, sizeof(tm));
  return true;
}

// (x0,x1) pass over nf = 4*nbatch fields
template <typename R>
wz_status launch_p01(wz_plan* pl, int kind, const P01Kern<R>& k, const P01Args<R>& args_in, int nb, int fmul = 1) {
  // args_in.I: inner volume the tiles run over (L2*L3, or L1*L2*L3 in the axis-0 kernel of the single-axis
  // decomposition); fmul: fields per (source, spin) (L0 in its axis-1 kernel)
  const int nseg_tiles = (int)(args_in.I / k.nseg), nf = 4 * nb * fmul;
  P01Args<R> args = args_in;
  args.rev = next_sweep(pl);
  // pass C launches spin-fastest: the four CTAs that share one phi tile run together (380 -> 360 us per launch
  // at 32^4 x 12); the same order slows pass E' (296 -> 346 us) and is not used there
  args.comp_fast = (kind == WZ_K_P01_MID) ? 1 : 0;
  args.tm_ahead = 0;
  if (pl->tile_prefetch && (kind == WZ_K_P01_MID || kind == WZ_K_P01_FWDCG)) {  // passes C and A' (wz_p01.cuh: E' does not gain)
    const int wave = wave_ctas(pl, (const void*)k.fn, k.nt, k.smem);
    if ((long)nseg_tiles * nf > 2L * wave &&  // at least two waves: something to run ahead of
        make_tile_tmap<R>(&args.tm_in, args.in, args_in.I, k.l0, k.l1, k.nseg, nf, k.half != 0))
      args.tm_ahead = wave;
  }
  {
    ProfScope ps(pl, kind);
    k.fn<<<dim3((unsigned)nseg_tiles, (unsigned)nf), k.nt, k.smem, pl->lstream>>>(args);
  }
  WZ_CUDA(cudaGetLastError());
  if (args.red.partials && k.split_finalize) {
    // the pass left one partial per CTA (4 spin components x tiles per source): total + scalar update
    const int nblk = 4 * nseg_tiles;
    ProfScope ps(pl, WZ_K_OTHER);
    switch (k.fin) {
      case FIN_PQ: k_finalize<FIN_PQ><<<nb, FINALIZE_NT, 0, pl->lstream>>>(args.red, nblk, args.gate); break;
      case FIN_RR: k_finalize<FIN_RR><<<nb, FINALIZE_NT, 0, pl->lstream>>>(args.red, nblk, args.gate); break;
      case FIN_RRS: k_finalize<FIN_RRS><<<nb, FINALIZE_NT, 0, pl->lstream>>>(args.red, nblk, args.gate); break;
      case FIN_PP: k_finalize<FIN_PP><<<nb, FINALIZE_NT, 0, pl->lstream>>>(args.red, nblk, args.gate); break;
      default: k_finalize<FIN_STORE><<<nb, FINALIZE_NT, 0, pl->lstream>>>(args.red, nblk, args.gate); break;
    }
    WZ_CUDA(cudaGetLastError());
  }
  return WZ_OK;
}

// One (x0,x1) pass in the mode `mk` names.  Two-axis tiles: one launch.  Single-axis decomposition (ws.p0s): the
// axis-0 kernel carries the mode (twist, site-local step, CG fusion) and plain axis-1 transforms run before it
// (inverse-type modes), after it (forward-type modes) or both (MID), in place on the FFT temporary, with every x0
// slice passed as a field of its own.  +2u of traffic per axis-1 launch, but every run is 512 bytes long.
// per-source partials of the reductions of the (x0,x1) passes: 4 spin components x tiles
template <typename R>
int partials_needed(const wz_plan* pl, const OpWS<R>& ws) {
  if (ws.p0s) return (int)((long)pl->L[1] * pl->I / ws.p0s->min_nseg()) * 4;
  return (int)(pl->I / ws.p01->min_nseg()) * 4;
}

enum { PASS_FWD_TYPE = 1, PASS_INV_TYPE = 2, PASS_MID_TYPE = 3 };
template <typename R>
wz_status pass01(wz_plan* pl, OpWS<R>& ws, int kind, P01Kern<R> P01Entry<R>::*mk, int type, const P01Args<R>& a, int nb) {
  if (!ws.p0s) return launch_p01<R>(pl, kind, ws.p01->*mk, a, nb);
  const int L0 = pl->L[0];
  wz_status s;
  P01Args<R> ax{};  // the axis-1 sub-pass: fields = (source, spin, x0), no twist, no scale
  ax.I = pl->I; ax.apbc = 0; ax.scale = R(1); ax.gate = a.gate; ax.fdiv = L0;
  if (type == PASS_INV_TYPE || type == PASS_MID_TYPE) {
    ax.in = a.in; ax.out = const_cast<cpx<R>*>(a.in);  // in place (a.in is the FFT temporary in these modes)
    if ((s = launch_p01<R>(pl, WZ_K_P01_INV, ws.p1s->inv, ax, nb, L0)) != WZ_OK) return s;
  }
  P01Args<R> a0 = a;
  a0.I = (long)pl->L[1] * pl->I;
  if ((s = launch_p01<R>(pl, kind, ws.p0s->*mk, a0, nb)) != WZ_OK) return s;
  if (type == PASS_FWD_TYPE || type == PASS_MID_TYPE) {
    ax.in = a.out; ax.out = a.out;
    if ((s = launch_p01<R>(pl, WZ_K_P01_FWD, ws.p1s->fwd, ax, nb, L0)) != WZ_OK) return s;
  }
  return WZ_OK;
}

// (x2,x3) pass over nb sources
template <typename R>
wz_status launch_p23(wz_plan* pl, int kind, const P23Entry<R>& e, void (*k)(const P23Args<R>),
                     const P23Args<R>& args, int nb) {
  const dim3 grid((unsigned)(pl->L[0] * pl->L[1]), (unsigned)nb, (unsigned)e.nhalf);
  P23Args<R> a2 = args;
  a2.rev = next_sweep(pl);
  const size_t smem = args.pc ? e.smem_pc : e.smem;
  a2.pf_dist = (int)((long)kPrefetchPercent * wave_ctas(pl, (const void*)k, e.nt, smem) / 100);
  if ((long)grid.x * grid.y <= a2.pf_dist) a2.pf_dist = 0;  // a single wave: nothing to run ahead of
  return launch<R>(pl, kind, k, grid, e.nt, smem, a2);
}
// Momentum-space multiply pass on the FFT temporary `cur`; in place, or into the other
// temporary where the kernel works on half the spin components per CTA.  `cur` follows.
template <typename R>
wz_status mult_pass(wz_plan* pl, OpWS<R>& ws, P23Args<R>& b, cpx<R>*& cur, int nb, cpx<R>* t = nullptr, cpx<R>* t2 = nullptr) {
  if (!t) { t = ws.t; t2 = ws.t2; }  // the two temporaries (whole batch, or the block a CG iteration works on)
  cpx<R>* dst = (ws.p23->nhalf == 2) ? ((cur == t) ? t2 : t) : cur;
  b.in = cur; b.out = dst;
  void (*kern)(const P23Args<R>) = b.pc ? ws.p23->multpc : ws.p23->mult;
  b.ctab = nullptr;
  if (!b.pc && ws.ctab && ws.ctab_rho == b.rho && ws.p23->multt) {  // c(p) from the table built for this rho
    kern = ws.p23->multt;
    b.ctab = ws.ctab;
  }
  wz_status s = launch_p23<R>(pl, WZ_K_P23_MULT, *ws.p23, kern, b, nb);
  // two components per CTA: the diagonal term of M0^-1 needs the pair the CTA does not hold -> second launch
  if (s == WZ_OK && b.pc && ws.p23->diagpc) s = launch_p23<R>(pl, WZ_K_P23_MULT, *ws.p23, ws.p23->diagpc, b, nb);
  cur = dst;
  return s;
}

RedArgs red_of(wz_plan* pl) {
  RedArgs r;
  r.partials = pl->partials; r.counter = pl->counter; r.st = pl->d_state; r.store = nullptr;
  r.pstride = pl->npartials;
  return r;
}

template <typename R>
OpWS<R>& ws_of(wz_plan* pl);
template <>
OpWS<float>& ws_of<float>(wz_plan* pl) { return pl->wsf; }
template <>
OpWS<double>& ws_of<double>(wz_plan* pl) { return pl->wsd; }

template <typename R>
OpParams<R> make_op(const double m[2], const double g[2], double rho, int dagger, int pc = 0) {
  OpParams<R> op;
  op.m_re = (R)m[0]; op.m_im = (R)m[1];
  op.g2_re = (R)(2.0 * g[0]); op.g2_im = (R)(2.0 * g[1]);
  op.rho = (R)rho; op.dagger = dagger; op.pc = pc; op.shift = R(0);
  return op;
}

// c(p) table of the multiply pass (wz_p23.cuh, P23_MULTT) for this rho: allocated on first use, rebuilt when rho
// changes.  Called at entry-point level only (never inside a stream capture); a pass launched while the table is
// missing or belongs to another rho computes c(p) on the fly as before.
template <typename R>
wz_status ensure_ctab(wz_plan* pl, OpWS<R>& ws, double rho) {
  if (pl->no_ctab || !ws.p23 || !ws.p23->multt) return WZ_OK;
  if (!ws.ctab && !dev_alloc(pl, &ws.ctab, (size_t)pl->V)) { ws.ctab = nullptr; cudaGetLastError(); return WZ_OK; }  // no memory: on the fly
  if (ws.ctab_rho == (R)rho) return WZ_OK;
  {
    ProfScope ps(pl, WZ_K_OTHER);
    const int grid = (int)std::min<long>((pl->V + CGK_NT - 1) / CGK_NT, 148L * 8);
    k_ctab<R><<<grid, CGK_NT, 0, pl->lstream>>>(ws.ctab, ws.tab, pl->L[0], pl->L[1], pl->L[2], pl->L[3], (R)rho);
  }
  WZ_CUDA(cudaGetLastError());
  ws.ctab_rho = (R)rho;
  return WZ_OK;
}

// ---- 4D FFT (steps a1, a2 / a4, a5) ---------------------------------------------
template <typename R>
wz_status fft4d_impl(wz_plan* pl, int direction, int apbc, const cpx<R>* in, cpx<R>* out, int nb) {
  OpWS<R>& ws = ws_of<R>(pl);
  P01Args<R> a{};
  a.I = pl->I; a.apbc = apbc; a.scale = R(1);
  P23Args<R> b{};
  b.nplanes = pl->L[0] * pl->L[1]; b.L1 = pl->L[1]; b.scale = R(1); b.tab = ws.tab;
  b.rho = R(1); b.sign = R(1);
  if (direction > 0) {
    a.in = in; a.out = out;
    wz_status s = pass01<R>(pl, ws, WZ_K_P01_FWD, &P01Entry<R>::fwd, PASS_FWD_TYPE, a, nb);
    if (s != WZ_OK) return s;
    b.in = out; b.out = out;
    return launch_p23<R>(pl, WZ_K_P23_FFT, *ws.p23, ws.p23->fwd, b, nb);
  }
  b.in = in; b.out = out;
  wz_status s = launch_p23<R>(pl, WZ_K_P23_FFT, *ws.p23, ws.p23->inv, b, nb);
  if (s != WZ_OK) return s;
  a.in = out; a.out = out; a.scale = (R)(1.0 / (double)pl->V);
  return pass01<R>(pl, ws, WZ_K_P01_INV, &P01Entry<R>::inv, PASS_INV_TYPE, a, nb);
}

// ---- out = M in or M^dag in: passes A, B, E --------------------------
template <typename R>
wz_status apply_M_impl(wz_plan* pl, int dagger, const cpx<R>* phi, const double m[2], const double g[2],
                       double rho, const cpx<R>* in, cpx<R>* out, int nb) {
  OpWS<R>& ws = ws_of<R>(pl);
  wz_status s = ensure_ctab<R>(pl, ws, rho);
  if (s != WZ_OK) return s;
  P01Args<R> a{};
  a.I = pl->I; a.apbc = 1; a.scale = R(1);
  a.in = in; a.out = ws.t;
  s = pass01<R>(pl, ws, WZ_K_P01_FWD, &P01Entry<R>::fwd, PASS_FWD_TYPE, a, nb);
  if (s != WZ_OK) return s;
  P23Args<R> b{};
  b.nplanes = pl->L[0] * pl->L[1]; b.L1 = pl->L[1]; b.scale = (R)(1.0 / (double)pl->V);
  b.tab = ws.tab; b.rho = (R)rho; b.sign = dagger ? R(-1) : R(1);
  cpx<R>* cur = ws.t;
  if ((s = mult_pass<R>(pl, ws, b, cur, nb)) != WZ_OK) return s;
  a.in = cur; a.out = cur;
  a.psi = in; a.phi = phi; a.site_out = out; a.op = make_op<R>(m, g, rho, dagger);
  return pass01<R>(pl, ws, WZ_K_P01_END, &P01Entry<R>::end, PASS_INV_TYPE, a, nb);
}

// ---- out = M^dag M in: passes A-E.  With `cg` set (nb = 1) the kernels are gated on
// the solve being active and pass C leaves alpha = rho/<p, A p> in the CG state. -----
template <typename R>
wz_status apply_MdagM_impl(wz_plan* pl, const cpx<R>* phi, const double m[2], const double g[2],
                           double rho, const cpx<R>* in, cpx<R>* out, int nb, bool cg, bool pc = false,
                           double sigma_pc = 0.0) {
  // sigma_pc (pc only): + sigma (M0^-1)^dag M0^-1, the operator of Eq. 7.14
  // pc: Mtilde^dag Mtilde with Mtilde = M M0^-1 = 1 + Y M0^-1: same five passes,
  // the multiply passes apply M0^-1 / (M0^-1)^dag, the site-local steps use Y alone
  OpWS<R>& ws = ws_of<R>(pl);
  const CGState* gate = cg ? pl->d_state : nullptr;
  const R invV = (R)(1.0 / (double)pl->V);
  wz_status s;
  if (!pc && (s = ensure_ctab<R>(pl, ws, rho)) != WZ_OK) return s;
  P01Args<R> a{};
  a.I = pl->I; a.apbc = 1; a.scale = R(1); a.gate = gate;
  a.in = in; a.out = ws.t;
  if ((s = pass01<R>(pl, ws, WZ_K_P01_FWD, &P01Entry<R>::fwd, PASS_FWD_TYPE, a, nb)) != WZ_OK) return s;  // A
  P23Args<R> b{};
  b.nplanes = pl->L[0] * pl->L[1]; b.L1 = pl->L[1]; b.scale = invV;
  b.tab = ws.tab; b.rho = (R)rho; b.sign = pc ? R(-1) : R(1); b.gate = gate;
  b.pc = pc ? 1 : 0; b.m_re = (R)m[0]; b.m_im = (R)m[1];
  cpx<R>* cur = ws.t;
  if ((s = mult_pass<R>(pl, ws, b, cur, nb)) != WZ_OK) return s;  // B
  a.in = cur; a.out = cur;
  a.psi = in; a.phi = phi; a.site_out = ws.chi; a.op = make_op<R>(m, g, rho, 0, pc);
  if (pc) a.op.shift = (R)sigma_pc;
  if (cg) {
    a.red = red_of(pl);
    if (partials_needed(pl, ws) > pl->npartials) return WZ_EINVAL;
    s = pass01<R>(pl, ws, WZ_K_P01_MID, &P01Entry<R>::mid_pq, PASS_MID_TYPE, a, nb);  // C
  } else {
    s = pass01<R>(pl, ws, WZ_K_P01_MID, &P01Entry<R>::mid, PASS_MID_TYPE, a, nb);
  }
  if (s != WZ_OK) return s;
  b.sign = pc ? R(1) : R(-1);
  b.pc = pc ? 2 : 0;
  if ((s = mult_pass<R>(pl, ws, b, cur, nb)) != WZ_OK) return s;  // D
  a.in = cur; a.out = cur;
  a.red = RedArgs{};
  a.psi = ws.chi; a.site_out = out; a.op = make_op<R>(m, g, rho, 1, pc);
  return pass01<R>(pl, ws, WZ_K_P01_END, &P01Entry<R>::end, PASS_INV_TYPE, a, nb);  // E
}

// ---- out = M0^-1 in (dagger = 0) or (M0^-1)^dag in, Eq. (7.11): forward FFT, the 4x4 free
// inverse at every momentum (multiply pass with pc), inverse FFT.  in == out allowed. -------
template <typename R>
wz_status apply_M0inv_impl(wz_plan* pl, int dagger, const double m[2], double rho, const cpx<R>* in,
                           cpx<R>* out, int nb) {
  OpWS<R>& ws = ws_of<R>(pl);
  wz_status s;
  P01Args<R> a{};
  a.I = pl->I; a.apbc = 1; a.scale = R(1);
  a.in = in; a.out = ws.t;
  if ((s = pass01<R>(pl, ws, WZ_K_P01_FWD, &P01Entry<R>::fwd, PASS_FWD_TYPE, a, nb)) != WZ_OK) return s;
  P23Args<R> b{};
  b.nplanes = pl->L[0] * pl->L[1]; b.L1 = pl->L[1]; b.scale = (R)(1.0 / (double)pl->V);
  b.tab = ws.tab; b.rho = (R)rho; b.sign = dagger ? R(1) : R(-1);
  b.pc = dagger ? 2 : 1; b.m_re = (R)m[0]; b.m_im = (R)m[1];
  cpx<R>* cur = ws.t;
  if ((s = mult_pass<R>(pl, ws, b, cur, nb)) != WZ_OK) return s;
  a.in = cur; a.out = out;  // 1/V already applied by the multiply pass
  return pass01<R>(pl, ws, WZ_K_P01_INV, &P01Entry<R>::inv, PASS_INV_TYPE, a, nb);
}

// ---- one CG iteration = five kernels: A' (x += alpha p pending from the
// previous iteration, p <- r + beta p, pass A), B, C (chi = M p, alpha = rho/||chi||^2),
// D, E' (q = M^dag chi in registers, r -= alpha q, ||r||^2 -> stop rule / beta /
// reliable-update request) = 18.5 u of traffic.  All scalars live in the device CG
// state; every kernel is gated on it.  x lags one update: flush_x() before x is used. --
template <typename R>
wz_status cg_iteration(wz_plan* pl, const cpx<R>* phi, const double m[2], const double g[2], double rho,
                       cpx<R>* r, cpx<R>* p, cpx<R>* x, int s0, int nb, bool pc, double sigma = 0.0) {
  // sources s0 .. s0 + nb - 1 of the batch (r, p, x: base pointers of the whole batch)
  // sigma != 0: the shifted system (M^dag M + sigma) x = b (Eq. 7.13): pass A' also
  // reduces <p,p> (alpha = rho / (||M p||^2 + sigma <p,p>)), pass E' uses q + sigma p
  // with pc the shift enters pass C instead (Eq. 7.14: + sigma (M0^-1)^dag M0^-1, see wz_p01.cuh)
  const bool sh = sigma != 0.0 && !pc;
  OpWS<R>& ws = ws_of<R>(pl);
  if (partials_needed(pl, ws) > pl->npartials) return WZ_EINVAL;
  const R invV = (R)(1.0 / (double)pl->V);
  const size_t off = (size_t)s0 * 4 * pl->V;  // first spinor of the block
  r += off; p += off; x += off;
  cpx<R>* const t = ws.t + off;
  cpx<R>* const t2 = ws.t2 ? ws.t2 + off : nullptr;
  cpx<R>* const chi = ws.chi + off;
  const CGState* gate = pl->d_state + s0;
  RedArgs red = red_of(pl);
  red.partials += (size_t)s0 * red.pstride; red.counter += s0; red.st += s0;
  wz_status s;
  P01Args<R> a{};
  a.I = pl->I; a.apbc = 1; a.scale = R(1); a.gate = gate;
  a.in = p; a.out = t; a.cg_r = r; a.cg_p = p; a.cg_x = x;
  if (sh) a.red = red;
  if ((s = pass01<R>(pl, ws, WZ_K_P01_FWDCG, sh ? &P01Entry<R>::fwdcg_s : &P01Entry<R>::fwdcg, PASS_FWD_TYPE, a, nb)) != WZ_OK) return s;
  P23Args<R> b{};
  b.nplanes = pl->L[0] * pl->L[1]; b.L1 = pl->L[1]; b.scale = invV;
  b.tab = ws.tab; b.rho = (R)rho; b.sign = pc ? R(-1) : R(1); b.gate = gate;
  b.pc = pc ? 1 : 0; b.m_re = (R)m[0]; b.m_im = (R)m[1];
  cpx<R>* cur = t;
  if ((s = mult_pass<R>(pl, ws, b, cur, nb, t, t2)) != WZ_OK) return s;
  a.in = cur; a.out = cur;
  a.psi = p; a.phi = phi; a.site_out = chi; a.op = make_op<R>(m, g, rho, 0, pc);
  if (pc) a.op.shift = (R)sigma;
  a.red = red;
  if ((s = pass01<R>(pl, ws, WZ_K_P01_MID, &P01Entry<R>::mid_pq, PASS_MID_TYPE, a, nb)) != WZ_OK) return s;
  b.sign = pc ? R(1) : R(-1);
  b.pc = pc ? 2 : 0;
  if ((s = mult_pass<R>(pl, ws, b, cur, nb, t, t2)) != WZ_OK) return s;
  a.in = cur; a.out = cur;
  a.psi = chi; a.site_out = nullptr; a.op = make_op<R>(m, g, rho, 1, pc);
  a.cg_r = r; a.cg_p = p; a.cg_x = x; a.op.shift = sh ? (R)sigma : R(0);
  return pass01<R>(pl, ws, WZ_K_P01_ENDCG, sh ? &P01Entry<R>::endcg_s : &P01Entry<R>::endcg, PASS_INV_TYPE, a, nb);
}

}  // namespace

// =============================== C ABI =========================================
extern "C" {

const char* wz_status_string(wz_status s) {
  switch (s) {
    case WZ_OK: return "ok";
    case WZ_EINVAL: return "invalid argument";
    case WZ_EUNSUPPORTED: return "unsupported lattice extents";
    case WZ_ENOMEM: return "out of device memory";
    case WZ_ECUDA: return "CUDA error";
    case WZ_ENOTCONVERGED: return "CG did not converge within max_iter";
  }
  return "unknown status";
}
const char* wz_last_error(void) { return g_err; }
const char* wz_version(void) { return "0.1"; }

int wz_supported(int T, int L1, int L2, int L3, wz_dtype dtype) {
  if (T < 2 || (T & 1)) return 0;
  const long I = (long)L2 * L3;
  // every plan needs the complex128 operator (reliable updates, true residual)
  const auto* ad = find_p01<double>(T, L1, I);
  const auto* bd = find_p23<double>(L2, L3);
  if (!ad || !bd || I % ad->nseg()) return 0;
  if (dtype == WZ_C64) {
    const auto* af = find_p01<float>(T, L1, I);
    const auto* bf = find_p23<float>(L2, L3);
    if (!af || !bf || I % af->nseg()) return 0;
  }
  return 1;
}

static void prof_collect(wz_plan* pl) {
  cudaStreamSynchronize(pl->stream);
  for (size_t i = 0; i < pl->prof_kind.size(); ++i) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, pl->prof_ev[2 * i], pl->prof_ev[2 * i + 1]) == cudaSuccess) {
      pl->prof_ms[pl->prof_kind[i]] += ms;
      pl->prof_n[pl->prof_kind[i]] += 1;
    }
    cudaEventDestroy(pl->prof_ev[2 * i]);
    cudaEventDestroy(pl->prof_ev[2 * i + 1]);
  }
  cudaGetLastError();
  pl->prof_ev.clear();
  pl->prof_kind.clear();
}

wz_status wz_plan_destroy(wz_plan* pl) {
  if (!pl) return WZ_EINVAL;
  WZ_ON_DEVICE(pl);
  prof_collect(pl);
  if (pl->iter_graph) cudaGraphExecDestroy(pl->iter_graph);
  if (pl->cap_stream) cudaStreamDestroy(pl->cap_stream);
  for (void* p : pl->allocs) cudaFree(p);
  if (pl->h_state) cudaFreeHost(pl->h_state);
  for (int i = 0; i < 2; ++i)
    if (pl->ev[i]) cudaEventDestroy(pl->ev[i]);
  delete pl;
  return WZ_OK;
}

wz_status wz_plan_create(wz_plan** plan, int T, int L1, int L2, int L3, wz_dtype dtype,
                         int max_batch, void* stream) {
  g_err[0] = 0;
  if (!plan) return WZ_EINVAL;
  *plan = nullptr;
  if (T < 2 || L1 < 2 || L2 < 2 || L3 < 2 || (T & 1) || max_batch < 1) return WZ_EINVAL;
  if (dtype != WZ_C64 && dtype != WZ_C128) return WZ_EINVAL;
  if (!wz_supported(T, L1, L2, L3, dtype)) return WZ_EUNSUPPORTED;
  int cur_dev = 0;
  WZ_CUDA(cudaGetDevice(&cur_dev));  // the plan lives on the current device (the one `stream` belongs to)
  if (!init_twiddles(cur_dev)) return WZ_ECUDA;
  wz_plan* pl = new (std::nothrow) wz_plan();
  if (!pl) return WZ_ENOMEM;
  pl->dev = cur_dev;
  pl->L[0] = T; pl->L[1] = L1; pl->L[2] = L2; pl->L[3] = L3;
  pl->I = (long)L2 * L3;
  pl->V = (long)T * L1 * pl->I;
  pl->dtype = dtype;
  pl->max_batch = max_batch;
  pl->stream = (cudaStream_t)stream;
  pl->lstream = pl->stream;
  memset(&pl->iter_key, 0, sizeof(pl->iter_key));
  {
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cur_dev) == cudaSuccess && sms > 0)
      pl->num_sms = sms;
    cudaGetLastError();
  }
  wz_status s = WZ_OK;
  const size_t n1 = (size_t)4 * pl->V;
  do {
    const size_t nbv = (size_t)max_batch * n1;  // CG vectors: one spinor per source
    if (dtype == WZ_C64) {
      if ((s = setup_ws<float>(pl, pl->wsf, max_batch)) != WZ_OK) break;
      if ((s = setup_ws<double>(pl, pl->wsd, 1)) != WZ_OK) break;
      float *r, *p, *xs;
      if (!dev_alloc(pl, &r, 2 * nbv) || !dev_alloc(pl, &p, 2 * nbv) || !dev_alloc(pl, &xs, 2 * nbv) ||
          !dev_alloc(pl, &pl->q128, n1) || !dev_alloc(pl, &pl->phi128, (size_t)pl->V)) { s = WZ_ENOMEM; break; }
      pl->r = r; pl->p = p; pl->xs = xs;
    } else {
      if ((s = setup_ws<double>(pl, pl->wsd, max_batch)) != WZ_OK) break;
      double *r, *p;
      if (!dev_alloc(pl, &r, 2 * nbv) || !dev_alloc(pl, &p, 2 * nbv) || !dev_alloc(pl, &pl->q128, n1)) {
        s = WZ_ENOMEM; break;
      }
      pl->r = r; pl->p = p;
    }
    // reduction workspace per source: a row of partials wide enough for every grid used
    long np = (pl->I / 2) * 4;
    if (np < 4096) np = 4096;
    if (pl->wsd.p01) np = std::max<long>(np, partials_needed(pl, pl->wsd));
    if (dtype == WZ_C64 && pl->wsf.p01) np = std::max<long>(np, partials_needed(pl, pl->wsf));
    pl->npartials = (int)np;
    if (!dev_alloc(pl, &pl->partials, (size_t)np * max_batch) || !dev_alloc(pl, &pl->counter, (size_t)max_batch) ||
        !dev_alloc(pl, &pl->d_state, (size_t)max_batch)) { s = WZ_ENOMEM; break; }
    if (!cuda_ok(cudaMemsetAsync(pl->counter, 0, max_batch * sizeof(unsigned), pl->stream), "cudaMemsetAsync") ||
        !cuda_ok(cudaMemsetAsync(pl->d_state, 0, max_batch * sizeof(CGState), pl->stream), "cudaMemsetAsync") ||
        !cuda_ok(cudaMallocHost((void**)&pl->h_state, 2 * max_batch * sizeof(CGState)), "cudaMallocHost") ||
        !cuda_ok(cudaEventCreateWithFlags(&pl->ev[0], cudaEventDisableTiming), "cudaEventCreate") ||
        !cuda_ok(cudaEventCreateWithFlags(&pl->ev[1], cudaEventDisableTiming), "cudaEventCreate") ||
        !cuda_ok(cudaStreamSynchronize(pl->stream), "cudaStreamSynchronize")) { s = WZ_ECUDA; break; }
  } while (0);
  if (s != WZ_OK) {
    wz_plan_destroy(pl);
    return s;
  }
  *plan = pl;
  return WZ_OK;
}

const char* wz_kind_name(int k) {
  static const char* names[WZ_NKINDS] = {"p01_fwd", "p23_mult", "p01_mid", "p01_end", "p23_fft",
                                         "p01_inv", "p01_fwdcg", "p01_endcg", "other"};
  return (k >= 0 && k < WZ_NKINDS) ? names[k] : "?";
}

wz_status wz_plan_profile(wz_plan* pl, int enable) {
  if (!pl) return WZ_EINVAL;
  WZ_ON_DEVICE(pl);
  prof_collect(pl);
  if (enable) {
    for (int k = 0; k < WZ_NKINDS; ++k) { pl->prof_ms[k] = 0.0; pl->prof_n[k] = 0; }
  }
  pl->profile = enable ? 1 : 0;
  return WZ_OK;
}

wz_status wz_plan_profile_read(wz_plan* pl, double* ms, unsigned long long* count) {
  if (!pl || !ms || !count) return WZ_EINVAL;
  WZ_ON_DEVICE(pl);
  prof_collect(pl);
  for (int k = 0; k < WZ_NKINDS; ++k) { ms[k] = pl->prof_ms[k]; count[k] = pl->prof_n[k]; }
  return WZ_OK;
}

wz_status wz_plan_set_block(wz_plan* pl, int sources_per_block) {
  if (!pl || sources_per_block < 0) return WZ_EINVAL;
  pl->block = sources_per_block;
  return WZ_OK;
}

wz_status wz_plan_set_graph(wz_plan* pl, int enable) {
  if (!pl) return WZ_EINVAL;
  pl->use_graph = enable ? 1 : 0;
  return WZ_OK;
}

int wz_plan_cg_history(const wz_plan* pl, int source, int* iterations, double* rel_residual, int cap) {
  if (!pl || source < 0 || source >= (int)pl->hist.size() || cap < 0) return -1;
  const auto& h = pl->hist[source];
  const int n = (int)h.size() < cap ? (int)h.size() : cap;
  for (int i = 0; i < n && iterations && rel_residual; ++i) { iterations[i] = h[i].first; rel_residual[i] = h[i].second; }
  return (int)h.size();
}

unsigned long long wz_plan_workspace_bytes(const wz_plan* pl) { return pl ? pl->bytes : 0ull; }
unsigned long long wz_plan_launch_count(const wz_plan* pl) { return pl ? pl->launches : 0ull; }
void wz_plan_reset_launch_count(wz_plan* pl) { if (pl) pl->launches = 0; }

wz_status wz_fft4d(wz_plan* pl, int direction, int antiperiodic_time, const void* in, void* out,
                   int nbatch) {
  g_err[0] = 0;
  if (!pl || !in || !out || (direction != 1 && direction != -1)) return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  const int ap = antiperiodic_time ? 1 : 0;
  if (pl->dtype == WZ_C64)
    return fft4d_impl<float>(pl, direction, ap, (const cpx<float>*)in, (cpx<float>*)out, nbatch);
  return fft4d_impl<double>(pl, direction, ap, (const cpx<double>*)in, (cpx<double>*)out, nbatch);
}

static wz_status check_op(const wz_plan* pl, const void* phi, const double* m, const double* g,
                          double rho, const void* in, const void* out, int nbatch) {
  if (!pl || !phi || !m || !g || !in || !out) return WZ_EINVAL;
  if (in == out) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0)) return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch) return WZ_EINVAL;
  return WZ_OK;
}

wz_status wz_apply_M(wz_plan* pl, int dagger, const void* phi, const double m[2], const double g[2],
                     double rho, const void* in, void* out, int nbatch) {
  g_err[0] = 0;
  wz_status s = check_op(pl, phi, m, g, rho, in, out, nbatch);
  if (s != WZ_OK) return s;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  const int dg = dagger ? 1 : 0;
  if (pl->dtype == WZ_C64)
    return apply_M_impl<float>(pl, dg, (const cpx<float>*)phi, m, g, rho, (const cpx<float>*)in,
                               (cpx<float>*)out, nbatch);
  return apply_M_impl<double>(pl, dg, (const cpx<double>*)phi, m, g, rho, (const cpx<double>*)in,
                              (cpx<double>*)out, nbatch);
}

wz_status wz_apply_MdagM(wz_plan* pl, const void* phi, const double m[2], const double g[2],
                         double rho, const void* in, void* out, int nbatch) {
  g_err[0] = 0;
  wz_status s = check_op(pl, phi, m, g, rho, in, out, nbatch);
  if (s != WZ_OK) return s;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  if (pl->dtype == WZ_C64)
    return apply_MdagM_impl<float>(pl, (const cpx<float>*)phi, m, g, rho, (const cpx<float>*)in,
                                   (cpx<float>*)out, nbatch, false);
  return apply_MdagM_impl<double>(pl, (const cpx<double>*)phi, m, g, rho, (const cpx<double>*)in,
                                  (cpx<double>*)out, nbatch, false);
}

}  // extern "C"

// =============================== CG driver ======================================
namespace {

constexpr int kCheckEvery = 8;  // iterations enqueued between two looks at the device state
constexpr double kDelta = 0.1;  // reliable-update threshold (G9)

int vec_grid(long n_real, int per_thread) {
  long nb = (n_real / per_thread + CGK_NT - 1) / CGK_NT;
  const long cap = 148L * 8;
  if (nb > cap) nb = cap;
  if (nb < 1) nb = 1;
  return (int)nb;
}

// All nb sources advance in lock step through the same five kernels per iteration
// (grid rows = sources), each with its own device-resident CG state: a source that
// has converged, hit max_iter or waits for a reliable update simply idles (its CTAs
// return at once).  The host looks at the states every kCheckEvery iterations, one
// chunk behind the GPU, and serves reliable updates source by source.
// R = iteration precision.  X: caller's complex128 solution buffer.
// pc: the preconditioned system of PAPER.md:900-921 (Eq. 7.8-7.10): btilde = (M0^-1)^dag b, CG on
// Mtilde^dag Mtilde xtilde = btilde with the stop rule on ITS residual (reading G15), x = M0^-1 xtilde;
// info.rel_residual_true is then ||b - M^dag M x|| / ||b|| of the original system.
template <typename R>
wz_status cg_batch(wz_plan* pl, const cpx<R>* phi, const cpx<R>* b, cpx<double>* X, const double m[2],
                   const double g[2], double rho, double tol, int max_iter, int nb, wz_cg_info* info,
                   bool pc, double sigma = 0.0, const double* tol_per_source = nullptr, bool reliable = true) {
  // tol_per_source (optional, nb entries): overrides tol source by source (defect-correction solves)
  // reliable = false (complex64 only): plain CG on the recursive residual, no reliable updates (the inner solver of
  // wz_cg_solve_dc); X still receives the float iterate folded into complex128 at exit
  // sigma: shift of the system (M^dag M + sigma) x = b (Eq. 7.13); with pc the system
  // iterated on is Eq. 7.14, (Mtilde^dag Mtilde + sigma (M0^-1)^dag M0^-1) xtilde = btilde
  constexpr bool kRU = (sizeof(R) == 4);
  constexpr int N = vec16<R>::N;
  const long n = 8 * pl->V;       // real entries of one spinor
  const size_t n1 = (size_t)4 * pl->V;  // complex entries of one spinor
  cudaStream_t st = pl->stream;
  R* r = (R*)pl->r; R* p = (R*)pl->p; R* xs = (R*)pl->xs;
  const int gv = vec_grid(n, N), gv2 = vec_grid(n, 2), gv4 = vec_grid(n, 4);
  wz_status s;
  if (!pc && (s = ensure_ctab<R>(pl, ws_of<R>(pl), rho)) != WZ_OK) return s;

  std::vector<CGState> h(nb);
  memset(h.data(), 0, sizeof(CGState) * nb);
  for (int j = 0; j < nb; ++j) {
    h[j].tol = tol_per_source ? tol_per_source[j] : tol; h[j].delta = kDelta; h[j].max_iter = max_iter; h[j].use_ru = (kRU && reliable) ? 1 : 0;
    h[j].true_rr = -1.0; h[j].shift = pc ? 0.0 : sigma;  // pc: the shift is inside pass C's reduction
    if (max_iter == 0) h[j].stop = 1;
  }
  WZ_CUDA(cudaMemcpyAsync(pl->d_state, h.data(), sizeof(CGState) * nb, cudaMemcpyHostToDevice, st));
  WZ_CUDA(cudaStreamSynchronize(st));  // h is pageable host memory
  if (!pc) {
    ProfScope ps(pl, WZ_K_OTHER);
    k_cg_init<R, R><<<dim3(gv2, nb), CGK_NT, 0, st>>>((const R*)b, r, p, kRU ? xs : nullptr, (double*)X, n, red_of(pl));
  } else if constexpr (kRU) {
    // btilde in complex128, source by source (the complex128 workspace holds one spinor)
    if (!pl->btilde128 && !dev_alloc(pl, &pl->btilde128, (size_t)pl->max_batch * n1)) return WZ_ENOMEM;
    for (int j = 0; j < nb; ++j) {
      {
        ProfScope ps(pl, WZ_K_OTHER);
        k_f2d<<<vec_grid(n, 1), CGK_NT, 0, st>>>((double*)pl->q128, (const float*)(b + j * n1), n);
      }
      if ((s = apply_M0inv_impl<double>(pl, 1, m, rho, pl->q128, pl->btilde128 + j * n1, 1)) != WZ_OK) return s;
    }
    ProfScope ps(pl, WZ_K_OTHER);
    k_cg_init<R, double><<<dim3(gv2, nb), CGK_NT, 0, st>>>((const double*)pl->btilde128, r, p, xs, (double*)X, n, red_of(pl));
  } else {
    if ((s = apply_M0inv_impl<R>(pl, 1, m, rho, b, (cpx<R>*)p, nb)) != WZ_OK) return s;  // btilde -> p
    ProfScope ps(pl, WZ_K_OTHER);
    k_cg_init<R, R><<<dim3(gv2, nb), CGK_NT, 0, st>>>((const R*)p, r, p, nullptr, (double*)X, n, red_of(pl));
  }
  WZ_CUDA(cudaGetLastError());

  // x += alpha p still pending from the last active iteration of source j (its kernels idle)
  auto flush_x = [&](int j) -> wz_status {
    {
      ProfScope ps(pl, WZ_K_OTHER);
      if constexpr (kRU) k_flush_x<R><<<dim3(gv, 1), CGK_NT, 0, st>>>(xs + j * n, p + j * n, n, pl->d_state + j);
      else k_flush_x<R><<<dim3(gv, 1), CGK_NT, 0, st>>>((R*)X + j * n, p + j * n, n, pl->d_state + j);
    }
    {
      ProfScope ps(pl, WZ_K_OTHER);
      k_clear_alpha<<<1, 1, 0, st>>>(pl->d_state + j);
    }
    WZ_CUDA(cudaGetLastError());
    return WZ_OK;
  };
  // residual of source j recomputed in complex128:  q128 = A X_j;  d = b_j - q128
  auto xsh = [&](int j) -> const double* { return (sigma != 0.0 && !pc) ? (const double*)(X + j * n1) : nullptr; };
  auto residual128 = [&](int j, bool update_r) -> wz_status {
    RedArgs ra = red_of(pl).for_source(j);
    struct Override {  // the one-source complex128 matvec is not part of the batched iteration
      wz_plan* p;
      explicit Override(wz_plan* q) : p(q) { p->prof_override = WZ_K_OTHER; }
      ~Override() { p->prof_override = -1; }
    } ov(pl);
    if constexpr (kRU) {
      if (update_r) {  // X += xs; xs = 0
        ProfScope ps(pl, WZ_K_OTHER);
        k_ru_accum<<<dim3(gv4, 1), CGK_NT, 0, st>>>((double*)(X + j * n1), (float*)(xs + j * n), n);
      }
      wz_status s2 = apply_MdagM_impl<double>(pl, pl->phi128, m, g, rho, X + j * n1, pl->q128, 1, false, pc, sigma);
      if (s2 != WZ_OK) return s2;
      ProfScope ps(pl, WZ_K_OTHER);
      if (pc) {  // rhs of the preconditioned system: btilde, kept in complex128
        const double* bt = (const double*)(pl->btilde128 + j * n1);
        if (update_r)
          k_resid<double, float, FIN_RU><<<dim3(gv2, 1), CGK_NT, 0, st>>>(bt, (const double*)pl->q128, (float*)(r + j * n), n, ra);
        else
          k_resid<double, float, FIN_TRUE><<<dim3(gv2, 1), CGK_NT, 0, st>>>(bt, (const double*)pl->q128, nullptr, n, ra);
      } else if (update_r)
        k_resid<float, float, FIN_RU><<<dim3(gv2, 1), CGK_NT, 0, st>>>(
            (const float*)(b + j * n1), (const double*)pl->q128, (float*)(r + j * n), n, ra, xsh(j), sigma);
      else
        k_resid<float, float, FIN_TRUE><<<dim3(gv2, 1), CGK_NT, 0, st>>>(
            (const float*)(b + j * n1), (const double*)pl->q128, nullptr, n, ra, xsh(j), sigma);
    } else {
      wz_status s2 = apply_MdagM_impl<double>(pl, (const cpx<double>*)phi, m, g, rho, X + j * n1, pl->q128, 1, false);
      if (s2 != WZ_OK) return s2;
      ProfScope ps(pl, WZ_K_OTHER);
      k_resid<double, double, FIN_TRUE><<<dim3(gv2, 1), CGK_NT, 0, st>>>(
          (const double*)(b + j * n1), (const double*)pl->q128, nullptr, n, ra, xsh(j), sigma);
    }
    WZ_CUDA(cudaGetLastError());
    return WZ_OK;
  };

  // One chunk = kCheckEvery iterations = 5 kCheckEvery launches with fixed arguments (every scalar lives in the
  // device CG state, every kernel is gated on it): captured once as a CUDA graph and replayed per chunk, so the
  // only host round trip of the solve is the lagged look at the states (north star iii).  Per-kernel
  // event timing (wz_plan_profile) needs stream launches and turns the graph off.
  // Sources advance in blocks of pl->block sources: each block runs its kCheckEvery iterations back to back, so
  // the vectors of a block are re-read by the next pass (and the next iteration) while they are still in the
  // 126 MB L2 instead of from HBM ("source blocks").  The sources are independent and every
  // reduction is per source, so the block size does not change any result.
  auto enqueue_chunk_plain = [&]() -> wz_status {
    const int blk = (pl->block > 0 && pl->block < nb) ? pl->block : nb;
    for (int s0 = 0; s0 < nb; s0 += blk) {
      const int nbk = (nb - s0 < blk) ? nb - s0 : blk;
      for (int it = 0; it < kCheckEvery; ++it) {
        wz_status s2;
        if constexpr (kRU)
          s2 = cg_iteration<R>(pl, phi, m, g, rho, (cpx<R>*)r, (cpx<R>*)p, (cpx<R>*)xs, s0, nbk, pc, sigma);
        else
          s2 = cg_iteration<R>(pl, phi, m, g, rho, (cpx<R>*)r, (cpx<R>*)p, (cpx<R>*)X, s0, nbk, pc, sigma);
        if (s2 != WZ_OK) return s2;
      }
    }
    return WZ_OK;
  };
  const bool graph = pl->use_graph && !pl->profile;
  if (graph) {
    IterGraphKey key;
    memset(&key, 0, sizeof(key));
    key.phi = phi; key.r = r; key.p = p; key.x = kRU ? (const void*)xs : (const void*)X;
    key.m[0] = m[0]; key.m[1] = m[1]; key.g[0] = g[0]; key.g[1] = g[1]; key.rho = rho; key.sigma = sigma;
    key.nb = nb; key.pc = pc ? 1 : 0; key.prec = (int)sizeof(R); key.block = pl->block;
    if (!pl->iter_graph || memcmp(&key, &pl->iter_key, sizeof(key)) != 0) {
      if (pl->iter_graph) { cudaGraphExecDestroy(pl->iter_graph); pl->iter_graph = nullptr; }
      if (!pl->cap_stream) WZ_CUDA(cudaStreamCreateWithFlags(&pl->cap_stream, cudaStreamNonBlocking));
      WZ_CUDA(cudaStreamBeginCapture(pl->cap_stream, cudaStreamCaptureModeThreadLocal));
      const unsigned long long l0 = pl->launches;
      const int sweep0 = pl->sweep;
      pl->lstream = pl->cap_stream;
      s = enqueue_chunk_plain();
      pl->lstream = pl->stream;
      pl->iter_graph_launches = (int)(pl->launches - l0);
      pl->launches = l0;
      pl->sweep = sweep0;
      cudaGraph_t gr = nullptr;
      cudaError_t ce = cudaStreamEndCapture(pl->cap_stream, &gr);
      if (s != WZ_OK) { if (gr) cudaGraphDestroy(gr); return s; }
      WZ_CUDA(ce);
      ce = cudaGraphInstantiate(&pl->iter_graph, gr, 0);
      cudaGraphDestroy(gr);
      WZ_CUDA(ce);
      pl->iter_key = key;
    }
  }
  auto enqueue_chunk = [&]() -> wz_status {
    if (!graph) return enqueue_chunk_plain();
    WZ_CUDA(cudaGraphLaunch(pl->iter_graph, st));
    pl->launches += pl->iter_graph_launches;
    return WZ_OK;
  };

  pl->hist.assign(nb, {});
  int slot_w = 0, slot_r = 0, inflight = 0;
  std::vector<int> ru_served(nb, 0);
  const CGState* snap = nullptr;
  for (;;) {
    while (inflight < 2) {
      if ((s = enqueue_chunk()) != WZ_OK) return s;
      WZ_CUDA(cudaMemcpyAsync(pl->h_state + slot_w * pl->max_batch, pl->d_state, sizeof(CGState) * nb,
                              cudaMemcpyDeviceToHost, st));
      WZ_CUDA(cudaEventRecord(pl->ev[slot_w], st));
      slot_w ^= 1;
      ++inflight;
    }
    WZ_CUDA(cudaEventSynchronize(pl->ev[slot_r]));
    snap = pl->h_state + slot_r * pl->max_batch;
    slot_r ^= 1;
    --inflight;
    bool all_done = true;
    for (int j = 0; j < nb; ++j) {
      auto& hj = pl->hist[j];
      if (snap[j].bnorm > 0.0 && (hj.empty() || hj.back().first != snap[j].iter))
        hj.emplace_back(snap[j].iter, std::sqrt(snap[j].need_ru ? snap[j].rr_new : snap[j].rr) / snap[j].bnorm);
      if (snap[j].converged || snap[j].stop) continue;
      all_done = false;
      if (snap[j].need_ru && snap[j].n_ru == ru_served[j]) {
        if ((s = flush_x(j)) != WZ_OK) return s;
        if ((s = residual128(j, true)) != WZ_OK) return s;  // sets beta; the next pass A' applies it
        ++ru_served[j];
      }
    }
    if (all_done) break;
  }
  WZ_CUDA(cudaStreamSynchronize(st));
  std::vector<CGState> fin(nb);
  WZ_CUDA(cudaMemcpy(fin.data(), pl->d_state, sizeof(CGState) * nb, cudaMemcpyDeviceToHost));
  for (int j = 0; j < nb; ++j) {
    if ((s = flush_x(j)) != WZ_OK) return s;
    if (fin[j].bnorm2 == 0.0) continue;
    if (!pc) {
      // true residual at exit: complex64 solves that converged carry it from their last
      // reliable update; everything else recomputes it now
      if (kRU && reliable && fin[j].converged) continue;
      if ((s = residual128(j, kRU)) != WZ_OK) return s;  // C64, not converged: fold xs into X first
      continue;
    }
    // preconditioned solve: X_j holds xtilde (+ xs still to be folded in for C64 solves that stopped)
    if constexpr (kRU) {
      if (!fin[j].converged) {
        ProfScope ps(pl, WZ_K_OTHER);
        k_ru_accum<<<dim3(gv4, 1), CGK_NT, 0, st>>>((double*)(X + j * n1), (float*)(xs + j * n), n);
      }
    }
    // x = M0^-1 xtilde in complex128, then the residual of the ORIGINAL system against b
    RedArgs ra = red_of(pl).for_source(j);
    if constexpr (kRU) {
      if ((s = apply_M0inv_impl<double>(pl, 0, m, rho, X + j * n1, X + j * n1, 1)) != WZ_OK) return s;
      if ((s = apply_MdagM_impl<double>(pl, pl->phi128, m, g, rho, X + j * n1, pl->q128, 1, false)) != WZ_OK) return s;
      ProfScope ps(pl, WZ_K_OTHER);
      k_resid<float, float, FIN_TRUE><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const float*)(b + j * n1), (const double*)pl->q128, nullptr, n, ra,
                                                                       sigma != 0.0 ? (const double*)(X + j * n1) : nullptr, sigma);
      k_norm2<float, FIN_AUX><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const float*)(b + j * n1), n, ra);
      pl->launches++;
    } else {
      if ((s = apply_M0inv_impl<double>(pl, 0, m, rho, X + j * n1, X + j * n1, 1)) != WZ_OK) return s;
      if ((s = apply_MdagM_impl<double>(pl, (const cpx<double>*)phi, m, g, rho, X + j * n1, pl->q128, 1, false)) != WZ_OK) return s;
      ProfScope ps(pl, WZ_K_OTHER);
      k_resid<double, double, FIN_TRUE><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const double*)(b + j * n1), (const double*)pl->q128, nullptr, n, ra,
                                                                         sigma != 0.0 ? (const double*)(X + j * n1) : nullptr, sigma);
      k_norm2<double, FIN_AUX><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const double*)(b + j * n1), n, ra);
      pl->launches++;
    }
    WZ_CUDA(cudaGetLastError());
  }
  WZ_CUDA(cudaStreamSynchronize(st));
  WZ_CUDA(cudaMemcpy(fin.data(), pl->d_state, sizeof(CGState) * nb, cudaMemcpyDeviceToHost));
  for (int j = 0; j < nb; ++j) {
    info[j].iterations = fin[j].iter;
    info[j].reliable_updates = ru_served[j];
    info[j].converged = fin[j].converged;
    info[j].rel_residual_recursive = fin[j].bnorm > 0 ? std::sqrt(fin[j].rr) / fin[j].bnorm : 0.0;
    const double bref = pc ? std::sqrt(fin[j].aux) : fin[j].bnorm;  // ||b|| of the system true_rr refers to
    info[j].rel_residual_true = bref > 0 ? std::sqrt(fin[j].true_rr < 0 ? 0.0 : fin[j].true_rr) / bref : 0.0;
  }
  return WZ_OK;
}

}  // namespace

// =============================== multi-shift CG =================================
namespace {

// All systems (M^dag M + sigma_i) x_i = b from one Krylov space (wz_cgk.cuh).  The base
// system -- the smallest shift -- runs through the five fused passes of cg_iteration (shifted passes A'/E' if
// its shift is not zero); two small kernels per iteration carry the other shifts along: k_ms_scalars (zeta
// recurrences, on the device) and k_ms_update (x_i, p_i; r read once for all shifts).  complex64 plans iterate
// without reliable updates (a recomputed residual would break the collinearity the method rests on) and
// then POLISH: per shift, the defect b - (A + sigma_i) x_i is formed in complex128 and solved for by the
// complex64 solver with reliable updates (wz_cg_solve_shift's loop), x_i += correction.
template <typename R>
wz_status ms_batch(wz_plan* pl, const cpx<R>* phi, const cpx<R>* b, cpx<double>* X, const double m[2],
                   const double g[2], double rho, const double* sigmas, int ns, double tol, int max_iter, int nb,
                   wz_cg_info* info) {
  constexpr bool kF = (sizeof(R) == 4);
  constexpr int N = vec16<R>::N;
  const long n = 8 * pl->V;
  const size_t n1 = (size_t)4 * pl->V;
  cudaStream_t st = pl->stream;
  R* r = (R*)pl->r; R* p = (R*)pl->p; R* xs = (R*)pl->xs;
  const int gv = vec_grid(n, N), gv2 = vec_grid(n, 2);
  wz_status s;
  int base = 0;
  for (int i = 1; i < ns; ++i)
    if (sigmas[i] < sigmas[base]) base = i;
  const double sigma0 = sigmas[base];
  if ((s = ensure_ctab<R>(pl, ws_of<R>(pl), rho)) != WZ_OK) return s;

  // workspace
  const size_t need = (size_t)ns * pl->max_batch;
  if (pl->ms_cap < need) {
    R* a = nullptr; R* c = nullptr;
    if (!dev_alloc(pl, &a, need * 2 * n1)) return WZ_ENOMEM;
    if (kF && !dev_alloc(pl, &c, need * 2 * n1)) return WZ_ENOMEM;
    pl->ms_p = a; pl->ms_x = c; pl->ms_cap = need;
  }
  if (!pl->ms_state && (!dev_alloc(pl, &pl->ms_state, (size_t)pl->max_batch) ||
                        !dev_alloc(pl, &pl->ms_true, (size_t)WZ_MAX_SHIFTS * pl->max_batch)))
    return WZ_ENOMEM;
  if (kF && !pl->ms_rhs) {
    R* a = nullptr;
    if (!dev_alloc(pl, &a, (size_t)pl->max_batch * 2 * n1)) return WZ_ENOMEM;
    pl->ms_rhs = a;
  }
  if (kF && !pl->ms_e && !dev_alloc(pl, &pl->ms_e, (size_t)pl->max_batch * n1)) return WZ_ENOMEM;
  R* msp = (R*)pl->ms_p;
  // x_i: complex128 plans write the caller's buffer directly; complex64 plans iterate on float copies
  R* msx_f = (R*)pl->ms_x;
  double* msx_d = (double*)X;
  // solution of the base system: advanced by pass A' (one update late) in its slot of the same array
  R* xbase_f = kF ? msx_f + (size_t)base * nb * n : nullptr;
  double* xbase_d = msx_d + (size_t)base * nb * n;

  std::vector<CGState> h(nb);
  memset(h.data(), 0, sizeof(CGState) * nb);
  for (int j = 0; j < nb; ++j) {
    h[j].tol = tol; h[j].delta = kDelta; h[j].max_iter = max_iter; h[j].use_ru = 0;
    h[j].true_rr = -1.0; h[j].shift = sigma0;
    if (max_iter == 0) h[j].stop = 1;
  }
  std::vector<MSState> hm(nb);
  memset(hm.data(), 0, sizeof(MSState) * nb);
  for (int j = 0; j < nb; ++j) {
    hm[j].nshift = ns; hm[j].alpha_prev = 1.0; hm[j].beta_prev = 0.0; hm[j].last_iter = 0;
    for (int i = 0; i < ns; ++i) { hm[j].zeta[i] = hm[j].zeta_prev[i] = 1.0; hm[j].srel[i] = sigmas[i] - sigma0; hm[j].rec[i] = 1.0; }
  }
  WZ_CUDA(cudaMemcpyAsync(pl->d_state, h.data(), sizeof(CGState) * nb, cudaMemcpyHostToDevice, st));
  WZ_CUDA(cudaMemcpyAsync(pl->ms_state, hm.data(), sizeof(MSState) * nb, cudaMemcpyHostToDevice, st));
  WZ_CUDA(cudaStreamSynchronize(st));
  {
    ProfScope ps(pl, WZ_K_OTHER);
    k_cg_init<R, R><<<dim3(gv2, nb), CGK_NT, 0, st>>>((const R*)b, r, p, nullptr, nullptr, n, red_of(pl));
  }
  {
    ProfScope ps(pl, WZ_K_OTHER);
    if constexpr (kF) k_ms_init<R, R, R><<<dim3(gv2, nb), CGK_NT, 0, st>>>((const R*)b, msp, msx_f, n, nb, ns);
    else k_ms_init<R, double, R><<<dim3(gv2, nb), CGK_NT, 0, st>>>((const R*)b, msp, msx_d, n, nb, ns);
  }
  WZ_CUDA(cudaGetLastError());

  int slot_w = 0, slot_r = 0, inflight = 0;
  const CGState* snap = nullptr;
  for (;;) {
    while (inflight < 2) {
      for (int it = 0; it < kCheckEvery; ++it) {
        if constexpr (kF) s = cg_iteration<R>(pl, phi, m, g, rho, (cpx<R>*)r, (cpx<R>*)p, (cpx<R>*)xbase_f, 0, nb, false, sigma0);
        else s = cg_iteration<R>(pl, phi, m, g, rho, (cpx<R>*)r, (cpx<R>*)p, (cpx<R>*)xbase_d, 0, nb, false, sigma0);
        if (s != WZ_OK) return s;
        if (ns > 1) {
          {
            ProfScope ps(pl, WZ_K_OTHER);
            k_ms_scalars<<<nb, WZ_MAX_SHIFTS, 0, st>>>(pl->ms_state, pl->d_state);
          }
          ProfScope ps(pl, WZ_K_OTHER);
          if constexpr (kF) k_ms_update<R, R><<<dim3(gv2, nb), CGK_NT, 0, st>>>(r, msp, msx_f, n, nb, base, pl->ms_state);
          else k_ms_update<R, double><<<dim3(gv2, nb), CGK_NT, 0, st>>>(r, msp, msx_d, n, nb, base, pl->ms_state);
        }
        WZ_CUDA(cudaGetLastError());
      }
      WZ_CUDA(cudaMemcpyAsync(pl->h_state + slot_w * pl->max_batch, pl->d_state, sizeof(CGState) * nb,
                              cudaMemcpyDeviceToHost, st));
      WZ_CUDA(cudaEventRecord(pl->ev[slot_w], st));
      slot_w ^= 1;
      ++inflight;
    }
    WZ_CUDA(cudaEventSynchronize(pl->ev[slot_r]));
    snap = pl->h_state + slot_r * pl->max_batch;
    slot_r ^= 1;
    --inflight;
    bool all_done = true;
    for (int j = 0; j < nb; ++j)
      if (!(snap[j].converged || snap[j].stop)) all_done = false;
    if (all_done) break;
  }
  WZ_CUDA(cudaStreamSynchronize(st));
  // the base system's x lags one update behind (pass A' applies it): flush
  {
    ProfScope ps(pl, WZ_K_OTHER);
    if constexpr (kF) k_flush_x<R><<<dim3(gv, nb), CGK_NT, 0, st>>>(xbase_f, p, n, pl->d_state);
    else k_flush_x<double><<<dim3(gv, nb), CGK_NT, 0, st>>>(xbase_d, (const double*)p, n, pl->d_state);
  }
  {
    ProfScope ps(pl, WZ_K_OTHER);
    k_clear_alpha<<<nb, 1, 0, st>>>(pl->d_state);
  }
  if constexpr (kF) {  // complex64 plans: x_i -> the caller's complex128 buffer
    ProfScope ps(pl, WZ_K_OTHER);
    k_to_double<float><<<vec_grid((long)ns * nb * n, 1), CGK_NT, 0, st>>>(msx_d, msx_f, (long)ns * nb * n, 0);
  }
  WZ_CUDA(cudaGetLastError());
  std::vector<CGState> fin(nb);
  std::vector<MSState> finm(nb);
  WZ_CUDA(cudaMemcpyAsync(fin.data(), pl->d_state, sizeof(CGState) * nb, cudaMemcpyDeviceToHost, st));
  WZ_CUDA(cudaMemcpyAsync(finm.data(), pl->ms_state, sizeof(MSState) * nb, cudaMemcpyDeviceToHost, st));
  WZ_CUDA(cudaStreamSynchronize(st));

  // true residuals ||b - (A + sigma_i) x_i||^2 in complex128, every shift and source
  const cpx<double>* phid = kF ? pl->phi128 : (const cpx<double>*)phi;
  auto true_residuals = [&](int i) -> wz_status {
    struct Override {
      wz_plan* p;
      explicit Override(wz_plan* q) : p(q) { p->prof_override = WZ_K_OTHER; }
      ~Override() { p->prof_override = -1; }
    } ov(pl);
    for (int j = 0; j < nb; ++j) {
      cpx<double>* xij = X + ((size_t)i * nb + j) * n1;
      wz_status s2 = apply_MdagM_impl<double>(pl, phid, m, g, rho, xij, pl->q128, 1, false);
      if (s2 != WZ_OK) return s2;
      RedArgs ra = red_of(pl).for_source(j);
      ra.store = pl->ms_true + (size_t)i * pl->max_batch + j;
      ProfScope ps(pl, WZ_K_OTHER);
      if constexpr (kF)  // also leaves the defect, rounded to complex64, as the right-hand side of the polishing solve
        k_resid<float, float, FIN_STORE><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const float*)(b + j * n1), (const double*)pl->q128,
                                                                          (float*)pl->ms_rhs + j * n, n, ra, (const double*)xij, sigmas[i]);
      else
        k_resid<double, double, FIN_STORE><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const double*)(b + j * n1), (const double*)pl->q128,
                                                                            nullptr, n, ra, (const double*)xij, sigmas[i]);
      WZ_CUDA(cudaGetLastError());
    }
    return WZ_OK;
  };
  std::vector<double> tr((size_t)WZ_MAX_SHIFTS * pl->max_batch, 0.0);
  auto read_true = [&]() -> wz_status {
    WZ_CUDA(cudaMemcpyAsync(tr.data(), pl->ms_true, sizeof(double) * tr.size(), cudaMemcpyDeviceToHost, st));
    WZ_CUDA(cudaStreamSynchronize(st));
    return WZ_OK;
  };
  for (int i = 0; i < ns; ++i) {
    if ((s = true_residuals(i)) != WZ_OK) return s;
    if ((s = read_true()) != WZ_OK) return s;
    for (int j = 0; j < nb; ++j) {
      wz_cg_info& o = info[(size_t)i * nb + j];
      const double bn = fin[j].bnorm;
      o.iterations = (i == base) ? fin[j].iter : finm[j].its[i];
      o.reliable_updates = 0;
      o.converged = (i == base) ? fin[j].converged : finm[j].frozen[i];
      if (bn == 0.0) o.converged = 1;
      o.rel_residual_recursive = bn > 0 ? ((i == base) ? std::sqrt(fin[j].rr) / bn : finm[j].rec[i]) : 0.0;
      o.rel_residual_true = bn > 0 ? std::sqrt(tr[(size_t)i * pl->max_batch + j]) / bn : 0.0;
    }
    if constexpr (kF) {
      // polish: solve (A + sigma_i) e = d_i for the sources whose true residual is above tol (complex64 drift)
      std::vector<double> tolj(nb, 0.5);
      bool any = false;
      for (int j = 0; j < nb; ++j) {
        const wz_cg_info& o = info[(size_t)i * nb + j];
        if (fin[j].bnorm > 0 && o.rel_residual_true > tol) {
          tolj[j] = 0.95 * tol / o.rel_residual_true;  // relative to ||d||: ends at 0.95 tol ||b||
          any = true;
        } else {
          tolj[j] = 1e30;  // nothing to do: converges at once
        }
      }
      if (any) {
        int spent = 0;
        for (int j = 0; j < nb; ++j) spent = std::max(spent, info[(size_t)i * nb + j].iterations);
        std::vector<wz_cg_info> pol(nb);
        s = cg_batch<float>(pl, (const cpx<float>*)phi, (const cpx<float>*)pl->ms_rhs, pl->ms_e, m, g, rho, tol,
                            std::max(0, max_iter - spent), nb, pol.data(), false, sigmas[i], tolj.data());
        if (s != WZ_OK) return s;
        {
          ProfScope ps(pl, WZ_K_OTHER);
          k_rat_term<double><<<dim3(gv2, nb), CGK_NT, 0, st>>>((double*)(X + (size_t)i * nb * n1), (const double*)pl->ms_e, 1.0, n, 0);
        }
        WZ_CUDA(cudaGetLastError());
        if ((s = true_residuals(i)) != WZ_OK) return s;
        if ((s = read_true()) != WZ_OK) return s;
        for (int j = 0; j < nb; ++j) {
          wz_cg_info& o = info[(size_t)i * nb + j];
          if (tolj[j] > 1e29) continue;
          o.iterations += pol[j].iterations;
          o.reliable_updates = pol[j].reliable_updates;
          o.rel_residual_true = std::sqrt(tr[(size_t)i * pl->max_batch + j]) / fin[j].bnorm;
          o.converged = (o.rel_residual_true <= tol * (1.0 + 1e-9)) ? 1 : 0;
        }
      }
    }
  }
  return WZ_OK;
}

}  // namespace

extern "C" wz_status wz_cg_solve_multishift(wz_plan* pl, const void* phi, const void* b, void* x, const double m[2],
                                            const double g[2], double rho, const double* sigmas, int nshift, double tol,
                                            int max_iter, int nbatch, wz_cg_info* info) {
  g_err[0] = 0;
  if (!pl || !phi || !b || !x || !m || !g || !info || !sigmas) return WZ_EINVAL;
  if (nshift < 1 || nshift > WZ_MAX_SHIFTS) return WZ_EINVAL;
  for (int i = 0; i < nshift; ++i)
    if (!(sigmas[i] >= 0.0)) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0) || !(tol > 0.0) || max_iter < 0) return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch || x == b) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  wz_status s;
  if (pl->dtype == WZ_C64) {
    const long nphi = 2 * pl->V;
    {
      ProfScope ps(pl, WZ_K_OTHER);
      k_f2d<<<vec_grid(nphi, 1), CGK_NT, 0, pl->stream>>>((double*)pl->phi128, (const float*)phi, nphi);
    }
    WZ_CUDA(cudaGetLastError());
    s = ms_batch<float>(pl, (const cpx<float>*)phi, (const cpx<float>*)b, (cpx<double>*)x, m, g, rho, sigmas, nshift,
                        tol, max_iter, nbatch, info);
  } else {
    s = ms_batch<double>(pl, (const cpx<double>*)phi, (const cpx<double>*)b, (cpx<double>*)x, m, g, rho, sigmas,
                         nshift, tol, max_iter, nbatch, info);
  }
  if (s != WZ_OK) return s;
  for (int i = 0; i < nshift * nbatch; ++i)
    if (!info[i].converged) return WZ_ENOTCONVERGED;
  return WZ_OK;
}

// =============================== defect correction ==============================
// complex128 outer loop around complex64 inner solves restarted at every step (oracle O9; PAPER.md:957;
// SURVEY 8(f) NEXT-3 "complex64 inner / complex128 outer").  WZ_C64 plans.
extern "C" wz_status wz_cg_solve_dc(wz_plan* pl, const void* phi_, const void* b_, void* x_, const double m[2],
                                    const double g[2], double rho, double tol, double inner_tol, int max_iter,
                                    int nbatch, wz_cg_info* info) {
  g_err[0] = 0;
  if (!pl || !phi_ || !b_ || !x_ || !m || !g || !info) return WZ_EINVAL;
  if (pl->dtype != WZ_C64) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0) || !(tol > 0.0) || !(inner_tol > 0.0 && inner_tol < 1.0) || max_iter < 0) return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch || x_ == b_) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  const int nb = nbatch;
  const long n = 8 * pl->V;
  const size_t n1 = (size_t)4 * pl->V;
  cudaStream_t st = pl->stream;
  const cpx<float>* phi = (const cpx<float>*)phi_;
  const cpx<float>* b = (const cpx<float>*)b_;
  cpx<double>* X = (cpx<double>*)x_;
  const int gv2 = vec_grid(n, 2);
  if (!pl->ms_true && !dev_alloc(pl, &pl->ms_true, (size_t)WZ_MAX_SHIFTS * pl->max_batch)) return WZ_ENOMEM;
  if (!pl->ms_rhs) {
    float* a = nullptr;
    if (!dev_alloc(pl, &a, (size_t)pl->max_batch * 2 * n1)) return WZ_ENOMEM;
    pl->ms_rhs = a;
  }
  if (!pl->ms_e && !dev_alloc(pl, &pl->ms_e, (size_t)pl->max_batch * n1)) return WZ_ENOMEM;
  {
    ProfScope ps(pl, WZ_K_OTHER);
    k_f2d<<<vec_grid(2 * pl->V, 1), CGK_NT, 0, st>>>((double*)pl->phi128, (const float*)phi, 2 * pl->V);
  }
  WZ_CUDA(cudaGetLastError());
  WZ_CUDA(cudaMemsetAsync(X, 0, sizeof(cpx<double>) * n1 * nb, st));
  std::vector<double> tr(nb, 0.0), bnorm(nb, 0.0), tolj(nb);
  std::vector<int> done(nb, 0), iters(nb, 0), outer(nb, 0);
  std::vector<wz_cg_info> inner(nb);
  for (;;) {
    {  // defects d_j = b_j - A X_j in complex128, rounded to complex64 as the inner right-hand sides
      struct Override {
        wz_plan* p;
        explicit Override(wz_plan* q) : p(q) { p->prof_override = WZ_K_OTHER; }
        ~Override() { p->prof_override = -1; }
      } ov(pl);
      for (int j = 0; j < nb; ++j) {
        if (done[j]) continue;
        wz_status s = apply_MdagM_impl<double>(pl, pl->phi128, m, g, rho, X + j * n1, pl->q128, 1, false);
        if (s != WZ_OK) return s;
        RedArgs ra = red_of(pl).for_source(j);
        ra.store = pl->ms_true + j;
        ProfScope ps(pl, WZ_K_OTHER);
        k_resid<float, float, FIN_STORE><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const float*)(b + j * n1), (const double*)pl->q128,
                                                                          (float*)pl->ms_rhs + j * n, n, ra);
        WZ_CUDA(cudaGetLastError());
      }
    }
    WZ_CUDA(cudaMemcpyAsync(tr.data(), pl->ms_true, sizeof(double) * nb, cudaMemcpyDeviceToHost, st));
    WZ_CUDA(cudaStreamSynchronize(st));
    bool all_done = true;
    int spent = 0;
    for (int j = 0; j < nb; ++j) {
      if (outer[j] == 0 && !done[j]) bnorm[j] = std::sqrt(tr[j]);  // X = 0: the defect is b itself
      if (!done[j] && (bnorm[j] == 0.0 || std::sqrt(tr[j]) <= tol * bnorm[j])) done[j] = 1;
      if (!done[j]) all_done = false;
      spent = std::max(spent, iters[j]);
    }
    if (all_done || spent >= max_iter) break;
    for (int j = 0; j < nb; ++j) tolj[j] = done[j] ? 1e30 : inner_tol;
    wz_status s = cg_batch<float>(pl, phi, (const cpx<float>*)pl->ms_rhs, pl->ms_e, m, g, rho, inner_tol, max_iter - spent,
                                  nb, inner.data(), false, 0.0, tolj.data(), false);
    if (s != WZ_OK) return s;
    for (int j = 0; j < nb; ++j) {
      if (done[j]) continue;
      ProfScope ps(pl, WZ_K_OTHER);
      k_rat_term<double><<<dim3(gv2, 1), CGK_NT, 0, st>>>((double*)(X + j * n1), (const double*)(pl->ms_e + j * n1), 1.0, n, 0);
      WZ_CUDA(cudaGetLastError());
      iters[j] += inner[j].iterations;
      outer[j] += 1;
    }
  }
  bool ok = true;
  for (int j = 0; j < nb; ++j) {
    info[j].iterations = iters[j];
    info[j].reliable_updates = outer[j];
    info[j].converged = done[j];
    info[j].rel_residual_true = bnorm[j] > 0 ? std::sqrt(tr[j]) / bnorm[j] : 0.0;
    info[j].rel_residual_recursive = info[j].rel_residual_true;
    if (!done[j]) ok = false;
  }
  return ok ? WZ_OK : WZ_ENOTCONVERGED;
}

// =============================== defect correction, binary16 storage =============================
// wz_cg_solve_dc_half (oracle O10): the outer loop of wz_cg_solve_dc, the inner solver with t, chi, r, p
// STORED as two binary16 values per complex number (arithmetic in float, reductions in double, x in float): 10.5u of
// traffic per iteration instead of 18.5u.  The defect is normalised to unit rms before each inner solve, so every stored
// value sits in binary16's normal range without per-vector scales.
namespace {

wz_status half_setup(wz_plan* pl, double rho) {
  OpWS<float>& w = pl->wsh;
  if (!w.p01) {
    w.p01 = find_p01<float>(pl->L[0], pl->L[1], pl->I, 1);
    w.p23 = find_p23<float>(pl->L[2], pl->L[3], 1);
    if (!w.p01 || !w.p23 || pl->I % w.p01->nseg()) { w.p01 = nullptr; return WZ_EUNSUPPORTED; }
    if (!set_smem_kern(w.p01->fwdcg) || !set_smem_kern(w.p01->mid_pq) || !set_smem_kern(w.p01->endcg) ||
        !set_smem(w.p23->mult, w.p23->smem) || !set_smem(w.p23->multt, w.p23->smem))
      return WZ_ECUDA;
    wave_ctas(pl, (const void*)w.p23->mult, w.p23->nt, w.p23->smem);
    wave_ctas(pl, (const void*)w.p23->multt, w.p23->nt, w.p23->smem);
    const size_t nel = (size_t)pl->max_batch * 4 * pl->V;  // complex numbers per batch of spinors, 4 bytes each
    unsigned *t = nullptr, *chi = nullptr, *r = nullptr, *p = nullptr;
    if (!dev_alloc(pl, &t, nel) || !dev_alloc(pl, &chi, nel) || !dev_alloc(pl, &r, nel) || !dev_alloc(pl, &p, nel)) {
      w.p01 = nullptr;
      return WZ_ENOMEM;
    }
    w.t = reinterpret_cast<cpx<float>*>(t);
    w.chi = reinterpret_cast<cpx<float>*>(chi);
    pl->h_r = r; pl->h_p = p;
    w.tab = pl->wsf.tab;
  }
  wz_status s = ensure_ctab<float>(pl, pl->wsf, rho);  // the complex64 operator's table serves both
  if (s != WZ_OK) return s;
  w.ctab = pl->wsf.ctab;
  w.ctab_rho = pl->wsf.ctab_rho;
  return WZ_OK;
}

// One CG iteration on the binary16-stored vectors: the same five passes as cg_iteration, all sources of the batch.
wz_status cg_iteration_half(wz_plan* pl, const cpx<float>* phi, const double m[2], const double g[2], double rho,
                            float* x, int nb) {
  typedef float R;
  OpWS<R>& ws = pl->wsh;
  if (partials_needed(pl, ws) > pl->npartials) return WZ_EINVAL;
  // The 1/V of the inverse transform is split: 1/(L0 L1) before the forward (x0,x1) transforms, 1/(L2 L3) in the multiply
  // pass.  Unnormalised, the temporary before pass E' holds the (x0,x1) transform of q = M^dag M p, whose entries reach
  // lambda_max * sqrt(L0 L1) = 1e5 ... 1e6 at 16^4 / 32^4: beyond binary16's largest finite value 65504.
  const R inv01 = (R)(1.0 / ((double)pl->L[0] * pl->L[1])), inv23 = (R)(1.0 / (double)pl->I);
  cpx<R>* const r = reinterpret_cast<cpx<R>*>(pl->h_r);  // cpxh storage behind cpx<R>-typed arguments: base pointers only
  cpx<R>* const p = reinterpret_cast<cpx<R>*>(pl->h_p);
  wz_status s;
  P01Args<R> a{};
  a.I = pl->I; a.apbc = 1; a.scale = inv01; a.gate = pl->d_state;
  a.in = p; a.out = ws.t; a.cg_r = r; a.cg_p = p; a.cg_x = reinterpret_cast<cpx<R>*>(x);
  if ((s = launch_p01<R>(pl, WZ_K_P01_FWDCG, ws.p01->fwdcg, a, nb)) != WZ_OK) return s;
  P23Args<R> b{};
  b.nplanes = pl->L[0] * pl->L[1]; b.L1 = pl->L[1]; b.scale = inv23;
  b.tab = ws.tab; b.rho = (R)rho; b.sign = R(1); b.gate = pl->d_state;
  b.pc = 0; b.m_re = (R)m[0]; b.m_im = (R)m[1];
  cpx<R>* cur = ws.t;
  if ((s = mult_pass<R>(pl, ws, b, cur, nb, ws.t, nullptr)) != WZ_OK) return s;
  a.in = cur; a.out = cur;
  a.psi = p; a.phi = phi; a.site_out = ws.chi; a.op = make_op<R>(m, g, rho, 0, 0);
  a.red = red_of(pl);
  // headroom for the temporaries of the second half: the one before pass E' holds the (x0,x1)-mode amplitudes of
  // q = M^dag M p, up to lambda_max / sqrt(L0 L1) times those of p (2500 |p| at 32^4, with |p| growing to tens in CG)
  constexpr float kHeadroom = 64.f;
  a.scale = inv01 / kHeadroom;
  if ((s = launch_p01<R>(pl, WZ_K_P01_MID, ws.p01->mid_pq, a, nb)) != WZ_OK) return s;
  a.scale = kHeadroom;  // pass E' multiplies it back after its inverse transform
  b.sign = R(-1);
  if ((s = mult_pass<R>(pl, ws, b, cur, nb, ws.t, nullptr)) != WZ_OK) return s;
  a.in = cur; a.out = cur;
  a.psi = ws.chi; a.site_out = nullptr; a.op = make_op<R>(m, g, rho, 1, 0);
  a.cg_r = r; a.cg_p = p; a.cg_x = reinterpret_cast<cpx<R>*>(x);
  return launch_p01<R>(pl, WZ_K_P01_ENDCG, ws.p01->endcg, a, nb);
}

}  // namespace

extern "C" wz_status wz_cg_solve_dc_half(wz_plan* pl, const void* phi_, const void* b_, void* x_, const double m[2],
                                         const double g[2], double rho, double tol, double inner_tol, int max_iter,
                                         int nbatch, wz_cg_info* info) {
  g_err[0] = 0;
  if (!pl || !phi_ || !b_ || !x_ || !m || !g || !info) return WZ_EINVAL;
  if (pl->dtype != WZ_C64) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0) || !(tol > 0.0) || !(inner_tol > 0.0 && inner_tol < 1.0) || max_iter < 0) return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch || x_ == b_) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  wz_status s = half_setup(pl, rho);
  if (s != WZ_OK) return s;
  const int nb = nbatch;
  const long n = 8 * pl->V;
  const size_t n1 = (size_t)4 * pl->V;
  cudaStream_t st = pl->stream;
  const cpx<float>* phi = (const cpx<float>*)phi_;
  const cpx<float>* b = (const cpx<float>*)b_;
  cpx<double>* X = (cpx<double>*)x_;
  float* xs = (float*)pl->xs;
  __half* r16 = (__half*)pl->h_r;
  __half* p16 = (__half*)pl->h_p;
  const int gv2 = vec_grid(n, 2), gv1 = vec_grid(n, 1);
  if (!pl->ms_true && !dev_alloc(pl, &pl->ms_true, (size_t)WZ_MAX_SHIFTS * pl->max_batch)) return WZ_ENOMEM;
  if (!pl->ms_rhs) {
    float* a = nullptr;
    if (!dev_alloc(pl, &a, (size_t)pl->max_batch * 2 * n1)) return WZ_ENOMEM;
    pl->ms_rhs = a;
  }
  {
    ProfScope ps(pl, WZ_K_OTHER);
    k_f2d<<<vec_grid(2 * pl->V, 1), CGK_NT, 0, st>>>((double*)pl->phi128, (const float*)phi, 2 * pl->V);
  }
  WZ_CUDA(cudaGetLastError());
  WZ_CUDA(cudaMemsetAsync(X, 0, sizeof(cpx<double>) * n1 * nb, st));
  std::vector<double> tr(nb, 0.0), bnorm(nb, 0.0), scale(nb, 1.0);
  std::vector<int> done(nb, 0), iters(nb, 0), outer(nb, 0);
  std::vector<CGState> h(nb);
  for (;;) {
    {  // defects d_j = b_j - A X_j in complex128, kept as float (the inner right-hand sides before normalisation)
      struct Override {
        wz_plan* p;
        explicit Override(wz_plan* q) : p(q) { p->prof_override = WZ_K_OTHER; }
        ~Override() { p->prof_override = -1; }
      } ov(pl);
      for (int j = 0; j < nb; ++j) {
        if (done[j]) continue;
        if ((s = apply_MdagM_impl<double>(pl, pl->phi128, m, g, rho, X + j * n1, pl->q128, 1, false)) != WZ_OK) return s;
        RedArgs ra = red_of(pl).for_source(j);
        ra.store = pl->ms_true + j;
        ProfScope ps(pl, WZ_K_OTHER);
        k_resid<float, float, FIN_STORE><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const float*)(b + j * n1), (const double*)pl->q128,
                                                                          (float*)pl->ms_rhs + j * n, n, ra);
        WZ_CUDA(cudaGetLastError());
      }
    }
    WZ_CUDA(cudaMemcpyAsync(tr.data(), pl->ms_true, sizeof(double) * nb, cudaMemcpyDeviceToHost, st));
    WZ_CUDA(cudaStreamSynchronize(st));
    bool all_done = true;
    int spent = 0;
    for (int j = 0; j < nb; ++j) {
      if (outer[j] == 0 && !done[j]) bnorm[j] = std::sqrt(tr[j]);  // X = 0: the defect is b itself
      if (!done[j] && (bnorm[j] == 0.0 || std::sqrt(tr[j]) <= tol * bnorm[j])) done[j] = 1;
      if (!done[j]) all_done = false;
      spent = std::max(spent, iters[j]);
    }
    if (all_done || spent >= max_iter) break;
    // inner solves: plain CG on the normalised defects, binary16 storage, all unfinished sources in lock step
    memset(h.data(), 0, sizeof(CGState) * nb);
    for (int j = 0; j < nb; ++j) {
      h[j].tol = inner_tol; h[j].delta = kDelta; h[j].max_iter = max_iter - spent; h[j].use_ru = 0; h[j].true_rr = -1.0;
      h[j].converged = done[j];
      scale[j] = done[j] ? 1.0 : std::sqrt((double)n / 2.0) / std::sqrt(tr[j]);  // unit rms per complex component pair
    }
    WZ_CUDA(cudaMemcpyAsync(pl->d_state, h.data(), sizeof(CGState) * nb, cudaMemcpyHostToDevice, st));
    WZ_CUDA(cudaStreamSynchronize(st));
    for (int j = 0; j < nb; ++j) {
      if (done[j]) continue;
      ProfScope ps(pl, WZ_K_OTHER);
      k_h_init<<<gv2, CGK_NT, 0, st>>>((const float*)pl->ms_rhs + j * n, r16 + j * n, p16 + j * n, xs + j * n, n, scale[j],
                                       red_of(pl).for_source(j));
      WZ_CUDA(cudaGetLastError());
    }
    int slot_w = 0, slot_r = 0, inflight = 0;
    for (;;) {
      while (inflight < 2) {
        for (int it = 0; it < kCheckEvery; ++it)
          if ((s = cg_iteration_half(pl, phi, m, g, rho, xs, nb)) != WZ_OK) return s;
        WZ_CUDA(cudaMemcpyAsync(pl->h_state + slot_w * pl->max_batch, pl->d_state, sizeof(CGState) * nb,
                                cudaMemcpyDeviceToHost, st));
        WZ_CUDA(cudaEventRecord(pl->ev[slot_w], st));
        slot_w ^= 1;
        ++inflight;
      }
      WZ_CUDA(cudaEventSynchronize(pl->ev[slot_r]));
      const CGState* snap = pl->h_state + slot_r * pl->max_batch;
      slot_r ^= 1;
      --inflight;
      bool fin = true;
      for (int j = 0; j < nb; ++j)
        if (!(snap[j].converged || snap[j].stop)) fin = false;
      if (fin) break;
    }
    WZ_CUDA(cudaStreamSynchronize(st));
    WZ_CUDA(cudaMemcpy(h.data(), pl->d_state, sizeof(CGState) * nb, cudaMemcpyDeviceToHost));
    {
      ProfScope ps(pl, WZ_K_OTHER);
      k_h_flush_x<<<dim3(gv2, nb), CGK_NT, 0, st>>>(xs, p16, n, pl->d_state);  // the x update still pending (idle sources: alpha = 0)
    }
    WZ_CUDA(cudaGetLastError());
    for (int j = 0; j < nb; ++j) {
      if (done[j]) continue;
      ProfScope ps(pl, WZ_K_OTHER);
      k_h_accum<<<gv1, CGK_NT, 0, st>>>((double*)(X + j * n1), xs + j * n, n, 1.0 / scale[j]);
      WZ_CUDA(cudaGetLastError());
      iters[j] += h[j].iter;
      outer[j] += 1;
    }
  }
  bool ok = true;
  for (int j = 0; j < nb; ++j) {
    info[j].iterations = iters[j];
    info[j].reliable_updates = outer[j];
    info[j].converged = done[j];
    info[j].rel_residual_true = bnorm[j] > 0 ? std::sqrt(tr[j]) / bnorm[j] : 0.0;
    info[j].rel_residual_recursive = info[j].rel_residual_true;
    if (!done[j]) ok = false;
  }
  return ok ? WZ_OK : WZ_ENOTCONVERGED;
}

// wz_cg_solve_half (oracle O11): binary16 storage of t, chi, r, p with complex128 RELIABLE UPDATES: the loop
// of wz_cg_solve for WZ_C64 plans (reading G9) on the system normalised to unit rms; at every update the vectors are
// rescaled to unit rms again, so they never leave binary16's normal range and the search direction survives.
extern "C" wz_status wz_cg_solve_half(wz_plan* pl, const void* phi_, const void* b_, void* x_, const double m[2],
                                      const double g[2], double rho, double tol, int max_iter, int nbatch,
                                      wz_cg_info* info) {
  g_err[0] = 0;
  if (!pl || !phi_ || !b_ || !x_ || !m || !g || !info) return WZ_EINVAL;
  if (pl->dtype != WZ_C64) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0) || !(tol > 0.0) || max_iter < 0) return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch || x_ == b_) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  wz_status s = half_setup(pl, rho);
  if (s != WZ_OK) return s;
  const int nb = nbatch;
  const long n = 8 * pl->V;
  const size_t n1 = (size_t)4 * pl->V;
  cudaStream_t st = pl->stream;
  const cpx<float>* phi = (const cpx<float>*)phi_;
  const cpx<float>* b = (const cpx<float>*)b_;
  cpx<double>* X = (cpx<double>*)x_;
  float* xs = (float*)pl->xs;
  __half* r16 = (__half*)pl->h_r;
  __half* p16 = (__half*)pl->h_p;
  const int gv2 = vec_grid(n, 2), gv1 = vec_grid(n, 1);
  if (!pl->ms_true && !dev_alloc(pl, &pl->ms_true, (size_t)WZ_MAX_SHIFTS * pl->max_batch)) return WZ_ENOMEM;
  if (!pl->ms_rhs) {
    float* a = nullptr;
    if (!dev_alloc(pl, &a, (size_t)pl->max_batch * 2 * n1)) return WZ_ENOMEM;
    pl->ms_rhs = a;
  }
  {
    ProfScope ps(pl, WZ_K_OTHER);
    k_f2d<<<vec_grid(2 * pl->V, 1), CGK_NT, 0, st>>>((double*)pl->phi128, (const float*)phi, 2 * pl->V);
  }
  WZ_CUDA(cudaGetLastError());
  WZ_CUDA(cudaMemsetAsync(X, 0, sizeof(cpx<double>) * n1 * nb, st));
  std::vector<double> tr(nb, 0.0), bnorm(nb, 0.0), scale(nb, 1.0), true_rel(nb, -1.0);
  {  // ||b_j||
    RedArgs ra = red_of(pl);
    ra.store = pl->ms_true;
    ProfScope ps(pl, WZ_K_OTHER);
    k_norm2<float, FIN_STORE><<<dim3(gv2, nb), CGK_NT, 0, st>>>((const float*)b, n, ra);
  }
  WZ_CUDA(cudaGetLastError());
  WZ_CUDA(cudaMemcpyAsync(tr.data(), pl->ms_true, sizeof(double) * nb, cudaMemcpyDeviceToHost, st));
  WZ_CUDA(cudaStreamSynchronize(st));
  std::vector<CGState> h(nb);
  memset(h.data(), 0, sizeof(CGState) * nb);
  for (int j = 0; j < nb; ++j) {
    bnorm[j] = std::sqrt(tr[j]);
    h[j].tol = tol; h[j].delta = kDelta; h[j].max_iter = max_iter; h[j].use_ru = 1; h[j].true_rr = -1.0;
    if (bnorm[j] == 0.0) { h[j].converged = 1; true_rel[j] = 0.0; }
    else scale[j] = std::sqrt((double)n / 2.0) / bnorm[j];
    if (max_iter == 0) h[j].stop = 1;
  }
  WZ_CUDA(cudaMemcpyAsync(pl->d_state, h.data(), sizeof(CGState) * nb, cudaMemcpyHostToDevice, st));
  WZ_CUDA(cudaStreamSynchronize(st));
  for (int j = 0; j < nb; ++j) {
    if (bnorm[j] == 0.0) continue;
    ProfScope ps(pl, WZ_K_OTHER);
    k_h_init<<<gv2, CGK_NT, 0, st>>>((const float*)b + j * n, r16 + j * n, p16 + j * n, xs + j * n, n, scale[j],
                                     red_of(pl).for_source(j));
    WZ_CUDA(cudaGetLastError());
  }
  // X_j += x_j / s_j (x cleared), then the defect of source j in complex128: float copy in ms_rhs, ||d||^2 on the host
  auto fold_and_defect = [&](int j) -> wz_status {
    {
      ProfScope ps(pl, WZ_K_OTHER);
      k_h_flush_x<<<dim3(gv2, 1), CGK_NT, 0, st>>>(xs + j * n, p16 + j * n, n, pl->d_state + j);
    }
    {
      ProfScope ps(pl, WZ_K_OTHER);
      k_clear_alpha<<<1, 1, 0, st>>>(pl->d_state + j);
    }
    {
      ProfScope ps(pl, WZ_K_OTHER);
      k_h_accum_clear<<<gv1, CGK_NT, 0, st>>>((double*)(X + j * n1), xs + j * n, n, 1.0 / scale[j]);
    }
    WZ_CUDA(cudaGetLastError());
    struct Override {
      wz_plan* p;
      explicit Override(wz_plan* q) : p(q) { p->prof_override = WZ_K_OTHER; }
      ~Override() { p->prof_override = -1; }
    } ov(pl);
    wz_status s2 = apply_MdagM_impl<double>(pl, pl->phi128, m, g, rho, X + j * n1, pl->q128, 1, false);
    if (s2 != WZ_OK) return s2;
    RedArgs ra = red_of(pl).for_source(j);
    ra.store = pl->ms_true + j;
    {
      ProfScope ps(pl, WZ_K_OTHER);
      k_resid<float, float, FIN_STORE><<<dim3(gv2, 1), CGK_NT, 0, st>>>((const float*)(b + j * n1), (const double*)pl->q128,
                                                                        (float*)pl->ms_rhs + j * n, n, ra);
    }
    WZ_CUDA(cudaGetLastError());
    WZ_CUDA(cudaMemcpyAsync(&tr[j], pl->ms_true + j, sizeof(double), cudaMemcpyDeviceToHost, st));
    WZ_CUDA(cudaStreamSynchronize(st));
    return WZ_OK;
  };
  int slot_w = 0, slot_r = 0, inflight = 0;
  std::vector<int> ru_served(nb, 0);
  for (;;) {
    while (inflight < 2) {
      for (int it = 0; it < kCheckEvery; ++it)
        if ((s = cg_iteration_half(pl, phi, m, g, rho, xs, nb)) != WZ_OK) return s;
      WZ_CUDA(cudaMemcpyAsync(pl->h_state + slot_w * pl->max_batch, pl->d_state, sizeof(CGState) * nb,
                              cudaMemcpyDeviceToHost, st));
      WZ_CUDA(cudaEventRecord(pl->ev[slot_w], st));
      slot_w ^= 1;
      ++inflight;
    }
    WZ_CUDA(cudaEventSynchronize(pl->ev[slot_r]));
    const CGState* snap = pl->h_state + slot_r * pl->max_batch;
    slot_r ^= 1;
    --inflight;
    bool all_done = true;
    for (int j = 0; j < nb; ++j) {
      if (snap[j].converged || snap[j].stop) continue;
      all_done = false;
      if (!(snap[j].need_ru && snap[j].n_ru == ru_served[j])) continue;
      if ((s = fold_and_defect(j)) != WZ_OK) return s;  // reliable update (G9), on the normalised system
      const double Rn = std::sqrt(tr[j]);
      ProfScope ps(pl, WZ_K_OTHER);
      if (Rn <= tol * bnorm[j]) {
        true_rel[j] = Rn / bnorm[j];
        k_h_patch<<<1, 1, 0, st>>>(pl->d_state + j, 1.0, 0.0, 1);
      } else {
        const double s_new = std::sqrt((double)n / 2.0) / Rn, f = s_new / scale[j];
        k_h_patch<<<1, 1, 0, st>>>(pl->d_state + j, f * f, s_new * bnorm[j], 0);
        k_h_rescale<<<gv2, CGK_NT, 0, st>>>((const float*)pl->ms_rhs + j * n, r16 + j * n, p16 + j * n, n, s_new, (float)f,
                                            red_of(pl).for_source(j));
        pl->launches++;
        scale[j] = s_new;
      }
      WZ_CUDA(cudaGetLastError());
      ++ru_served[j];
    }
    if (all_done) break;
  }
  WZ_CUDA(cudaStreamSynchronize(st));
  WZ_CUDA(cudaMemcpy(h.data(), pl->d_state, sizeof(CGState) * nb, cudaMemcpyDeviceToHost));
  bool ok = true;
  for (int j = 0; j < nb; ++j) {
    if (true_rel[j] < 0.0) {  // stopped at max_iter: fold what there is, recompute the residual
      if ((s = fold_and_defect(j)) != WZ_OK) return s;
      true_rel[j] = std::sqrt(tr[j]) / bnorm[j];
    }
    info[j].iterations = h[j].iter;
    info[j].reliable_updates = ru_served[j];
    info[j].converged = h[j].converged;
    info[j].rel_residual_recursive = h[j].bnorm > 0 ? std::sqrt(h[j].rr) / h[j].bnorm : 0.0;
    info[j].rel_residual_true = true_rel[j];
    if (!h[j].converged) ok = false;
  }
  return ok ? WZ_OK : WZ_ENOTCONVERGED;
}

static wz_status cg_solve_any(wz_plan* pl, const void* phi, const void* b, void* x, const double m[2],
                              const double g[2], double rho, double tol, int max_iter, int nbatch,
                              wz_cg_info* info, bool pc, double sigma = 0.0) {
  g_err[0] = 0;
  if (!(sigma >= 0.0)) return WZ_EINVAL;
  if (!pl || !phi || !b || !x || !m || !g || !info) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0) || !(tol > 0.0) || max_iter < 0) return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch) return WZ_EINVAL;
  if (pc && m[0] == 0.0 && m[1] == 0.0) return WZ_EINVAL;  // M0 must be invertible at every momentum
  if (x == b) return WZ_EINVAL;  // b is re-read by every reliable update and for the true residual
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  wz_status s;
  if (pl->dtype == WZ_C64) {
    const long nphi = 2 * pl->V;
    {
      ProfScope ps(pl, WZ_K_OTHER);
      k_f2d<<<vec_grid(nphi, 1), CGK_NT, 0, pl->stream>>>((double*)pl->phi128, (const float*)phi, nphi);
    }
    WZ_CUDA(cudaGetLastError());
    s = cg_batch<float>(pl, (const cpx<float>*)phi, (const cpx<float>*)b, (cpx<double>*)x, m, g, rho, tol,
                        max_iter, nbatch, info, pc, sigma);
  } else {
    s = cg_batch<double>(pl, (const cpx<double>*)phi, (const cpx<double>*)b, (cpx<double>*)x, m, g, rho, tol,
                         max_iter, nbatch, info, pc, sigma);
  }
  if (s != WZ_OK) return s;
  for (int j = 0; j < nbatch; ++j)
    if (!info[j].converged) return WZ_ENOTCONVERGED;
  return WZ_OK;
}

extern "C" {

wz_status wz_cg_solve(wz_plan* pl, const void* phi, const void* b, void* x, const double m[2],
                      const double g[2], double rho, double tol, int max_iter, int nbatch, wz_cg_info* info) {
  return cg_solve_any(pl, phi, b, x, m, g, rho, tol, max_iter, nbatch, info, false);
}

wz_status wz_cg_solve_shift(wz_plan* pl, const void* phi, const void* b, void* x, const double m[2],
                            const double g[2], double rho, double sigma, double tol, int max_iter, int nbatch,
                            wz_cg_info* info) {
  return cg_solve_any(pl, phi, b, x, m, g, rho, tol, max_iter, nbatch, info, false, sigma);
}

wz_status wz_cg_solve_pc(wz_plan* pl, const void* phi, const void* b, void* x, const double m[2],
                         const double g[2], double rho, double tol, int max_iter, int nbatch, wz_cg_info* info) {
  return cg_solve_any(pl, phi, b, x, m, g, rho, tol, max_iter, nbatch, info, true);
}

wz_status wz_cg_solve_shift_pc(wz_plan* pl, const void* phi, const void* b, void* x, const double m[2],
                               const double g[2], double rho, double sigma, double tol, int max_iter, int nbatch,
                               wz_cg_info* info) {
  return cg_solve_any(pl, phi, b, x, m, g, rho, tol, max_iter, nbatch, info, true, sigma);
}

// Eq. (7.6)-(7.7) with the cutoff rule of PAPER.md:948: one CG solve per shift ("for each i"),
// preconditioned (Eq. 7.14) up to pc_cutoff, plain (Eq. 7.13) above; terms summed in complex128.
wz_status wz_rational_apply(wz_plan* pl, const void* phi, const void* eta, void* out, const double m[2],
                            const double g[2], double rho, double alpha0, const double* alphas,
                            const double* betas, int nshift, double pc_cutoff, double tol, int max_iter,
                            int nbatch, wz_cg_info* info) {
  g_err[0] = 0;
  if (!pl || !phi || !eta || !out || !m || !g || !info || nshift < 0 || (nshift > 0 && (!alphas || !betas)))
    return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch) return WZ_EINVAL;
  for (int i = 0; i < nshift; ++i)
    if (!(betas[i] >= 0.0)) return WZ_EINVAL;
  if (out == eta) return WZ_EINVAL;  // eta is the right-hand side of every shift
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  const size_t n1 = (size_t)4 * pl->V;
  const long n = 8 * pl->V;
  if (pl->ratX_cap < (size_t)pl->max_batch) {
    if (!dev_alloc(pl, &pl->ratX, (size_t)pl->max_batch * n1)) return WZ_ENOMEM;
    pl->ratX_cap = pl->max_batch;
  }
  const int gv2 = vec_grid(n, 2);
  {
    ProfScope ps(pl, WZ_K_OTHER);
    if (pl->dtype == WZ_C64)
      k_rat_term<float><<<dim3(gv2, nbatch), CGK_NT, 0, pl->stream>>>((double*)out, (const float*)eta, alpha0, n, 1);
    else
      k_rat_term<double><<<dim3(gv2, nbatch), CGK_NT, 0, pl->stream>>>((double*)out, (const double*)eta, alpha0, n, 1);
  }
  WZ_CUDA(cudaGetLastError());
  bool all_ok = true;
  for (int i = 0; i < nshift; ++i) {
    const bool pc = betas[i] <= pc_cutoff && !(m[0] == 0.0 && m[1] == 0.0);
    wz_status s = cg_solve_any(pl, phi, eta, pl->ratX, m, g, rho, tol, max_iter, nbatch, info + (size_t)i * nbatch,
                               pc, betas[i]);
    if (s == WZ_ENOTCONVERGED) all_ok = false;
    else if (s != WZ_OK) return s;
    ProfScope ps(pl, WZ_K_OTHER);
    k_rat_term<double><<<dim3(gv2, nbatch), CGK_NT, 0, pl->stream>>>((double*)out, (const double*)pl->ratX, alphas[i], n, 0);
    WZ_CUDA(cudaGetLastError());
  }
  WZ_CUDA(cudaStreamSynchronize(pl->stream));
  return all_ok ? WZ_OK : WZ_ENOTCONVERGED;
}

// Eq. (7.6)-(7.7) with ONE multi-shift solve for every shift above pc_cutoff (all of them if pc_cutoff < 0 or
// m = 0) and the paper's preconditioned per-shift solves (Eq. 7.14) below it.
wz_status wz_rational_apply_multishift(wz_plan* pl, const void* phi, const void* eta, void* out, const double m[2],
                                       const double g[2], double rho, double alpha0, const double* alphas,
                                       const double* betas, int nshift, double pc_cutoff, double tol, int max_iter,
                                       int nbatch, wz_cg_info* info) {
  g_err[0] = 0;
  if (!pl || !phi || !eta || !out || !m || !g || !info || nshift < 0 || (nshift > 0 && (!alphas || !betas)))
    return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch) return WZ_EINVAL;
  for (int i = 0; i < nshift; ++i)
    if (!(betas[i] >= 0.0)) return WZ_EINVAL;
  if (out == eta) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  const size_t n1 = (size_t)4 * pl->V;
  const long n = 8 * pl->V;
  std::vector<int> ms_idx, pc_idx;
  for (int i = 0; i < nshift; ++i) {
    const bool pc = betas[i] <= pc_cutoff && !(m[0] == 0.0 && m[1] == 0.0);
    (pc ? pc_idx : ms_idx).push_back(i);
  }
  if ((int)ms_idx.size() > WZ_MAX_SHIFTS) return WZ_EINVAL;
  const size_t needX = std::max<size_t>(ms_idx.size(), 1) * pl->max_batch;
  if (pl->ratX_cap < needX) {
    if (!dev_alloc(pl, &pl->ratX, needX * n1)) return WZ_ENOMEM;
    pl->ratX_cap = needX;
  }
  const int gv2 = vec_grid(n, 2);
  {
    ProfScope ps(pl, WZ_K_OTHER);
    if (pl->dtype == WZ_C64)
      k_rat_term<float><<<dim3(gv2, nbatch), CGK_NT, 0, pl->stream>>>((double*)out, (const float*)eta, alpha0, n, 1);
    else
      k_rat_term<double><<<dim3(gv2, nbatch), CGK_NT, 0, pl->stream>>>((double*)out, (const double*)eta, alpha0, n, 1);
  }
  WZ_CUDA(cudaGetLastError());
  bool all_ok = true;
  for (int i : pc_idx) {
    wz_status s = cg_solve_any(pl, phi, eta, pl->ratX, m, g, rho, tol, max_iter, nbatch, info + (size_t)i * nbatch,
                               true, betas[i]);
    if (s == WZ_ENOTCONVERGED) all_ok = false;
    else if (s != WZ_OK) return s;
    ProfScope ps(pl, WZ_K_OTHER);
    k_rat_term<double><<<dim3(gv2, nbatch), CGK_NT, 0, pl->stream>>>((double*)out, (const double*)pl->ratX, alphas[i], n, 0);
    WZ_CUDA(cudaGetLastError());
  }
  if (!ms_idx.empty()) {
    std::vector<double> sig(ms_idx.size());
    for (size_t k = 0; k < ms_idx.size(); ++k) sig[k] = betas[ms_idx[k]];
    std::vector<wz_cg_info> inf(ms_idx.size() * nbatch);
    wz_status s = wz_cg_solve_multishift(pl, phi, eta, pl->ratX, m, g, rho, sig.data(), (int)sig.size(), tol, max_iter,
                                         nbatch, inf.data());
    if (s == WZ_ENOTCONVERGED) all_ok = false;
    else if (s != WZ_OK) return s;
    for (size_t k = 0; k < ms_idx.size(); ++k) {
      for (int j = 0; j < nbatch; ++j) info[(size_t)ms_idx[k] * nbatch + j] = inf[k * nbatch + j];
      ProfScope ps(pl, WZ_K_OTHER);
      k_rat_term<double><<<dim3(gv2, nbatch), CGK_NT, 0, pl->stream>>>(
          (double*)out, (const double*)(pl->ratX + k * nbatch * n1), alphas[ms_idx[k]], n, 0);
      WZ_CUDA(cudaGetLastError());
    }
  }
  WZ_CUDA(cudaStreamSynchronize(pl->stream));
  return all_ok ? WZ_OK : WZ_ENOTCONVERGED;
}

wz_status wz_apply_M0inv(wz_plan* pl, int dagger, const double m[2], double rho, const void* in, void* out,
                         int nbatch) {
  g_err[0] = 0;
  if (!pl || !m || !in || !out) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0) || (m[0] == 0.0 && m[1] == 0.0)) return WZ_EINVAL;
  if (nbatch < 0 || nbatch > pl->max_batch) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  if (pl->dtype == WZ_C64)
    return apply_M0inv_impl<float>(pl, dagger ? 1 : 0, m, rho, (const cpx<float>*)in, (cpx<float>*)out, nbatch);
  return apply_M0inv_impl<double>(pl, dagger ? 1 : 0, m, rho, (const cpx<double>*)in, (cpx<double>*)out, nbatch);
}

// Dslash = the fermion matrix at m = 0, g = 0 (Eq. 2.19): passes A, B, E with a zero site-local term.
wz_status wz_apply_Dslash(wz_plan* pl, double rho, const void* in, void* out, int nbatch) {
  g_err[0] = 0;
  if (!pl || !in || !out || in == out) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0) || nbatch < 0 || nbatch > pl->max_batch) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  const double zero[2] = {0.0, 0.0};
  // the site-local coefficient m + 2 g phi vanishes identically; `in` (finite values) stands in for phi
  if (pl->dtype == WZ_C64)
    return apply_M_impl<float>(pl, 0, (const cpx<float>*)in, zero, zero, rho, (const cpx<float>*)in,
                               (cpx<float>*)out, nbatch);
  return apply_M_impl<double>(pl, 0, (const cpx<double>*)in, zero, zero, rho, (const cpx<double>*)in,
                              (cpx<double>*)out, nbatch);
}

wz_status wz_locality_profile(wz_plan* pl, double rho, int spin, double* f_host, int nf) {
  g_err[0] = 0;
  int rmax = 0;
  if (pl) for (int mu = 0; mu < 4; ++mu) rmax += pl->L[mu] / 2;
  if (!pl || !f_host || spin < 0 || spin > 3 || nf != rmax + 1 || !(rho > 0.0 && rho < 2.0)) return WZ_EINVAL;
  WZ_ON_DEVICE(pl);
  const size_t n1 = (size_t)4 * pl->V;
  const bool f32 = pl->dtype == WZ_C64;
  const size_t esz = f32 ? sizeof(cpx<float>) : sizeof(cpx<double>);
  void* eta = f32 ? (void*)pl->wsf.chi : (void*)pl->wsd.chi;  // plan temporaries: eta -> chi, psi -> r
  void* psi = pl->r;
  unsigned long long* d_f = reinterpret_cast<unsigned long long*>(pl->partials);  // >= 4096 doubles
  if (nf > pl->npartials) return WZ_EINVAL;
  WZ_CUDA(cudaMemsetAsync(eta, 0, n1 * esz, pl->stream));
  WZ_CUDA(cudaMemsetAsync(d_f, 0, sizeof(double) * nf, pl->stream));
  if (f32) {
    const cpx<float> one = {1.f, 0.f};
    WZ_CUDA(cudaMemcpyAsync((cpx<float>*)eta + (size_t)spin * pl->V, &one, sizeof(one), cudaMemcpyHostToDevice, pl->stream));
  } else {
    const cpx<double> one = {1.0, 0.0};
    WZ_CUDA(cudaMemcpyAsync((cpx<double>*)eta + (size_t)spin * pl->V, &one, sizeof(one), cudaMemcpyHostToDevice, pl->stream));
  }
  WZ_CUDA(cudaStreamSynchronize(pl->stream));  // `one` lives on this stack frame
  wz_status s = wz_apply_Dslash(pl, rho, eta, psi, 1);
  if (s != WZ_OK) return s;
  {
    ProfScope ps(pl, WZ_K_OTHER);
    const int grid = vec_grid(pl->V, 1);
    if (f32) k_locality<float><<<grid, CGK_NT, 0, pl->stream>>>((const cpx<float>*)psi, d_f, pl->L[0], pl->L[1], pl->L[2], pl->L[3]);
    else k_locality<double><<<grid, CGK_NT, 0, pl->stream>>>((const cpx<double>*)psi, d_f, pl->L[0], pl->L[1], pl->L[2], pl->L[3]);
  }
  WZ_CUDA(cudaGetLastError());
  WZ_CUDA(cudaMemcpyAsync(f_host, d_f, sizeof(double) * nf, cudaMemcpyDeviceToHost, pl->stream));
  WZ_CUDA(cudaStreamSynchronize(pl->stream));
  for (int r = 0; r < nf; ++r) f_host[r] = std::sqrt(f_host[r]);
  return WZ_OK;
}

wz_status wz_apply_MtdagMt(wz_plan* pl, const void* phi, const double m[2], const double g[2], double rho,
                           const void* in, void* out, int nbatch) {
  g_err[0] = 0;
  wz_status s = check_op(pl, phi, m, g, rho, in, out, nbatch);
  if (s != WZ_OK) return s;
  if (m[0] == 0.0 && m[1] == 0.0) return WZ_EINVAL;
  if (nbatch == 0) return WZ_OK;
  WZ_ON_DEVICE(pl);
  if (pl->dtype == WZ_C64)
    return apply_MdagM_impl<float>(pl, (const cpx<float>*)phi, m, g, rho, (const cpx<float>*)in,
                                   (cpx<float>*)out, nbatch, false, true);
  return apply_MdagM_impl<double>(pl, (const cpx<double>*)phi, m, g, rho, (const cpx<double>*)in,
                                  (cpx<double>*)out, nbatch, false, true);
}

}  // extern "C"

// =============================== no-allocation entry point =======================
// wz_apply_MdagM_noalloc: M^dag M without a plan and without any device allocation, for callers that cannot call
// cudaMalloc (code under CUDA graph capture, tight serving loops).  The matvec's scratch -- the FFT temporary t,
// chi = M psi, and the momentum tables -- lives in ONE file-scope device array of WZ_NOALLOC_MAX_BYTES (+ 4 KB of
// tables) that every GPU loading the library holds until exit.  All calls share it: calls that overlap on the GPU
// race.  Nothing in it has to start at zero: every byte a call reads is written earlier in the same call.
namespace {

constexpr size_t kNoAllocTabBytes = 4096;  // momentum tables [2][4][64], double at most
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocTabBytes + WZ_NOALLOC_MAX_BYTES];

// Per device: the DEVICE address of g_noalloc_scratch.  In host code the array's name is only a host-side stand-in
// for the symbol, never a device address: cudaGetSymbolAddress (with that device current) gives the address.
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mu;
unsigned char* g_noalloc_ptr[kNoAllocMaxDevices] = {nullptr};

wz_status noalloc_setup(int dev, unsigned char** ptr) {
  if (dev < 0 || dev >= kNoAllocMaxDevices) return WZ_EINVAL;
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    if (!init_twiddles(dev)) return WZ_ECUDA;  // __constant__ twiddle tables of the kernel modules, once per device
    unsigned char* p = nullptr;
    WZ_CUDA(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch));
    if (!p) { snprintf(g_err, sizeof(g_err), "cudaGetSymbolAddress(g_noalloc_scratch) gave a null address"); return WZ_ECUDA; }
    g_noalloc_ptr[dev] = p;
  }
  *ptr = g_noalloc_ptr[dev];
  return WZ_OK;
}

// Momentum tables (as setup_ws computes them on the host), written by the device straight into the head of the
// scratch array: device code may name the array directly.  tab[0][mu][n] = sin p_mu, tab[1][mu][n] = sin^2(p_mu/2),
// p_0 = 2 pi (n + 1/2)/T, p_i = 2 pi n/L_i; sinpi() reduces the argument exactly.
template <typename R>
__global__ void k_noalloc_tables(int L0, int L1, int L2, int L3) {
  R* tab = reinterpret_cast<R*>(g_noalloc_scratch);
  const int L[4] = {L0, L1, L2, L3};
  for (int i = threadIdx.x; i < 2 * 4 * 64; i += blockDim.x) {
    const int which = i / 256, mu = (i / 64) % 4, n = i % 64;
    double v = 0.0;
    if (n < L[mu]) {
      const double x = 2.0 * ((double)n + (mu == 0 ? 0.5 : 0.0)) / (double)L[mu];  // p / pi
      if (which == 0) {
        v = sinpi(x);
      } else {
        const double s = sinpi(0.5 * x);
        v = s * s;
      }
    }
    tab[i] = (R)v;
  }
}

template <typename R>
wz_status noalloc_MdagM(int T, int L1, int L2, int L3, const void* phi, const double m[2], const double g[2],
                        double rho, const void* in, void* out, int nb, cudaStream_t stream, int dev,
                        unsigned char* scratch) {
  // A plan object on the host stack: lattice, stream, kernel choices; its "workspace" points into the static array.
  wz_plan pl;
  pl.L[0] = T; pl.L[1] = L1; pl.L[2] = L2; pl.L[3] = L3;
  pl.I = (long)L2 * L3;
  pl.V = (long)T * L1 * pl.I;
  pl.dtype = (sizeof(R) == 4) ? WZ_C64 : WZ_C128;
  pl.max_batch = nb;
  pl.stream = stream; pl.lstream = stream;
  pl.dev = dev;
  pl.no_ctab = 1;  // no device allocation here: c(p) on the fly
  memset(&pl.iter_key, 0, sizeof(pl.iter_key));
  int sms = 0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0) pl.num_sms = sms;
  OpWS<R>& ws = ws_of<R>(&pl);
  ws.p01 = find_p01<R>(T, L1, pl.I);
  ws.p23 = find_p23<R>(L2, L3);
  if (!ws.p01 || !ws.p23 || pl.I % ws.p01->nseg()) return WZ_EUNSUPPORTED;
  if (T * L1 > 2048) {  // single-axis decomposition, as setup_ws chooses it
    const auto* e0 = find_p01<R>(T, 1, 0);
    const auto* e1 = find_p01<R>(L1, 1, 0);
    if (e0 && e1 && ((long)L1 * pl.I) % e0->nseg() == 0 && pl.I % e1->nseg() == 0) { ws.p0s = e0; ws.p1s = e1; }
  }
  // scratch: [tables 4 KB][t][t2 where the multiply pass is out of place][chi], nb spinors each
  const size_t u = (size_t)4 * pl.V * sizeof(cpx<R>);
  const int nvec = 2 + (ws.p23->nhalf == 2 ? 1 : 0);
  const size_t need = (size_t)nvec * nb * u;
  if (need > (size_t)WZ_NOALLOC_MAX_BYTES) {
    snprintf(g_err, sizeof(g_err), "wz_apply_MdagM_noalloc: this call needs %zu bytes of scratch (%d temporaries x %d "
             "sources x %zu bytes per spinor), the static array holds WZ_NOALLOC_MAX_BYTES = %zu",
             need, nvec, nb, u, (size_t)WZ_NOALLOC_MAX_BYTES);
    return WZ_EINVAL;
  }
  const P01Entry<R>* entries[3] = {ws.p01, ws.p0s, ws.p1s};
  for (const P01Entry<R>* e : entries) {
    if (!e) continue;
    if (!set_smem_kern(e->fwd) || !set_smem_kern(e->inv) || !set_smem_kern(e->mid) || !set_smem_kern(e->end)) return WZ_ECUDA;
  }
  if (!set_smem(ws.p23->mult, ws.p23->smem)) return WZ_ECUDA;
  ws.tab = reinterpret_cast<R*>(scratch);
  unsigned char* vec = scratch + kNoAllocTabBytes;
  ws.t = reinterpret_cast<cpx<R>*>(vec);
  if (nvec == 3) ws.t2 = reinterpret_cast<cpx<R>*>(vec + (size_t)nb * u);
  ws.chi = reinterpret_cast<cpx<R>*>(vec + (size_t)(nvec - 1) * nb * u);
  k_noalloc_tables<R><<<1, 256, 0, stream>>>(T, L1, L2, L3);
  WZ_CUDA(cudaGetLastError());
  return apply_MdagM_impl<R>(&pl, (const cpx<R>*)phi, m, g, rho, (const cpx<R>*)in, (cpx<R>*)out, nb, false);
}

}  // namespace

extern "C" wz_status wz_apply_MdagM_noalloc(int T, int L1, int L2, int L3, wz_dtype dtype, const void* phi,
                                            const double m[2], const double g[2], double rho, const void* in,
                                            void* out, int nbatch, void* stream) {
  g_err[0] = 0;
  if (!phi || !m || !g || !in || !out || in == out) return WZ_EINVAL;
  if (T < 2 || L1 < 2 || L2 < 2 || L3 < 2 || (T & 1) || nbatch < 0) return WZ_EINVAL;
  if (dtype != WZ_C64 && dtype != WZ_C128) return WZ_EINVAL;
  if (!(rho > 0.0 && rho < 2.0)) return WZ_EINVAL;
  if (!wz_supported(T, L1, L2, L3, dtype)) return WZ_EUNSUPPORTED;
  if (nbatch == 0) return WZ_OK;
  int dev = 0;
  WZ_CUDA(cudaGetDevice(&dev));  // works on the CURRENT device: `stream` and every pointer must belong to it
  unsigned char* scratch = nullptr;
  wz_status s = noalloc_setup(dev, &scratch);
  if (s != WZ_OK) return s;
  if (dtype == WZ_C64)
    return noalloc_MdagM<float>(T, L1, L2, L3, phi, m, g, rho, in, out, nbatch, (cudaStream_t)stream, dev, scratch);
  return noalloc_MdagM<double>(T, L1, L2, L3, phi, m, g, rho, in, out, nbatch, (cudaStream_t)stream, dev, scratch);
}
