// wz_kmod.cu -- instantiates the pass kernels.  Compiled once per module, -DWZ_MOD=0..7
// (paper_1005_3276_b200/build.py), so that the modules build in parallel:
//   0: (x0,x1) passes, complex64, 32x32 tiles specialised for 32^4 (BASELINE.json config 4)
//   1: (x0,x1) passes, complex64, the other large tiles (48x24, 64x64, 64x32)
//   2: (x0,x1) passes, complex64, small and generic tiles
//   3: (x0,x1) passes, complex128, benchmark lattices
//   4: (x0,x1) passes, complex128, the rest
//   5: (x2,x3) passes, complex64
//   6: (x2,x3) passes, complex128
//   7: binary16-storage variants (complex64 arithmetic): CG-fused (x0,x1) passes and the multiply pass
#include "wz_tables.cuh"

#ifndef WZ_MOD
#error "compile with -DWZ_MOD=<0..7>"
#endif

namespace wz {
namespace {

bool upload_twiddles(const void* tf, const void* td) {
  return cudaMemcpyToSymbol(c_twf, tf, sizeof(float2) * TWN) == cudaSuccess &&
         cudaMemcpyToSymbol(c_twd, td, sizeof(double2) * TWN) == cudaSuccess;
}

void p01f([[maybe_unused]] std::vector<P01Entry<float>>& v) {
  using R = float;
#if WZ_MOD == 0
  v.push_back(make_p01<R, 32, 32, 1024>());
#elif WZ_MOD == 1
  v.push_back(make_p01<R, 48, 24, 576>());
  v.push_back(make_p01<R, 64, 64, 4096>());
  v.push_back(make_p01<R, 64, 64>());
  v.push_back(make_p01<R, 64, 32>());
  v.push_back(make_p01<R, 64, 1>());  // single-axis passes of the 64x64 lattices (wz_lib.cu: pass01)
#elif WZ_MOD == 2
  v.push_back(make_p01<R, 4, 4>());
  v.push_back(make_p01<R, 8, 8>());
  v.push_back(make_p01<R, 8, 4>());
  v.push_back(make_p01<R, 16, 16>());
  v.push_back(make_p01<R, 32, 32>());
  v.push_back(make_p01<R, 48, 24>());
  v.push_back(make_p01<R, 32, 8>());
  v.push_back(make_p01<R, 32, 16>());
#elif WZ_MOD == 7
  v.push_back(make_p01_half<32, 32, 1024>());
  v.push_back(make_p01_half<8, 8>());
  v.push_back(make_p01_half<16, 16>());
  v.push_back(make_p01_half<32, 32>());
  v.push_back(make_p01_half<48, 24, 576>());
#endif
}
void p01d([[maybe_unused]] std::vector<P01Entry<double>>& v) {
  using R = double;
#if WZ_MOD == 3
  v.push_back(make_p01<R, 32, 32, 1024>());
  v.push_back(make_p01<R, 48, 24, 576>());
  v.push_back(make_p01<R, 64, 64, 4096>());
  v.push_back(make_p01<R, 64, 1>());  // single-axis passes of the 64x64 lattices (wz_lib.cu: pass01)
#elif WZ_MOD == 4
  v.push_back(make_p01<R, 4, 4>());
  v.push_back(make_p01<R, 8, 8>());
  v.push_back(make_p01<R, 8, 4>());
  v.push_back(make_p01<R, 16, 16>());
  v.push_back(make_p01<R, 32, 32>());
  v.push_back(make_p01<R, 48, 24>());
  v.push_back(make_p01<R, 64, 64>());
  v.push_back(make_p01<R, 32, 8>());
  v.push_back(make_p01<R, 32, 16>());
  v.push_back(make_p01<R, 64, 32>());
#endif
}
void p23f([[maybe_unused]] std::vector<P23Entry<float>>& v) {
#if WZ_MOD == 5
  using R = float;
  v.push_back(make_p23<R, 4, 4>());
  v.push_back(make_p23<R, 8, 8>());
  v.push_back(make_p23<R, 16, 8>());
  v.push_back(make_p23<R, 16, 16>());
  v.push_back(make_p23<R, 32, 32>());
  v.push_back(make_p23<R, 24, 24>());
  v.push_back(make_p23<R, 64, 64, 2>());  // one component pair per CTA (67 KB): three CTAs per SM instead of one
#endif
#if WZ_MOD == 7
  v.push_back(make_p23_half<8, 8>());
  v.push_back(make_p23_half<16, 16>());
  v.push_back(make_p23_half<32, 32>());
  v.push_back(make_p23_half<24, 24>());
#endif
}
void p23d([[maybe_unused]] std::vector<P23Entry<double>>& v) {
#if WZ_MOD == 6
  using R = double;
  v.push_back(make_p23<R, 4, 4>());
  v.push_back(make_p23<R, 8, 8>());
  v.push_back(make_p23<R, 16, 8>());
  v.push_back(make_p23<R, 16, 16>());
  v.push_back(make_p23<R, 32, 32>());
  v.push_back(make_p23<R, 24, 24>());
  // four 64x64 complex128 planes (266 KB) exceed one SM's shared memory: two per CTA there
  v.push_back(make_p23<R, 64, 64, 2>());
#endif
}

const KernelModule kModule = {upload_twiddles, p01f, p01d, p23f, p23d};

}  // namespace

#define WZ_CAT2(a, b) a##b
#define WZ_CAT(a, b) WZ_CAT2(a, b)
const KernelModule* WZ_CAT(wz_kernel_module_, WZ_MOD)() { return &kModule; }

}  // namespace wz
