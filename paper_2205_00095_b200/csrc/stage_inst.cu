// stage_inst.cu -- instantiations of the fused stage kernel for one (ndim, EOS, Riemann flux) triple
// and every order p = 0..4; compiled once per triple (-DDG_INST_ND=1|2|3 -DDG_INST_EOS=0|1
// -DDG_INST_RS=0|1) so that the translation units build in parallel.  Exports a launcher and a per-device preparation call,
// declared in dgrhd.cu.
#include "stage_kernel.cuh"

#ifndef DG_INST_ND
#error "compile with -DDG_INST_ND=... -DDG_INST_EOS=... -DDG_INST_RS=..."
#endif

#define DG_CAT_(a, b, c, d) a##b##_##c##d
#define DG_CAT(a, b, c, d) DG_CAT_(a, b, c, d)
#define DG_LAUNCH_NAME DG_CAT(dg_launch_stage_, DG_INST_ND, DG_INST_EOS, DG_INST_RS)
#define DG_PREPARE_NAME DG_CAT(dg_prepare_stage_, DG_INST_ND, DG_INST_EOS, DG_INST_RS)

// Shared-memory opt-in of the kernel on the CURRENT device (the attribute is per device; called by
// dgrhd_create, outside any stream capture).
template <int N>
static cudaError_t prepare_n() {
  using TS = TileShape<DG_INST_ND, N>;
  auto k = dg_stage_kernel<DG_INST_ND, N, DG_INST_EOS, DG_INST_RS>;
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, TS::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}

template <int N>
static cudaError_t launch_n(const StageArgs& a, cudaStream_t st) {
  using TS = TileShape<DG_INST_ND, N>;
  const long long ntx = (a.ne[0] + TS::TX - 1) / TS::TX, nty = (a.ne[1] + TS::TY - 1) / TS::TY,
                  ntz = (a.ne[2] + TS::TZ - 1) / TS::TZ;
  if (ntx <= 0 || nty <= 0 || ntz <= 0 || ntx > 2147483647LL || nty > 65535 || ntz > 65535)
    return cudaErrorInvalidConfiguration;
  dg_stage_kernel<DG_INST_ND, N, DG_INST_EOS, DG_INST_RS>
      <<<dim3((unsigned)ntx, (unsigned)nty, (unsigned)ntz), TS::NT, TS::SMEM_BYTES, st>>>(a);
  return cudaGetLastError();
}

cudaError_t DG_PREPARE_NAME(int N) {
  switch (N) {
    case 1: return prepare_n<1>();
    case 2: return prepare_n<2>();
    case 3: return prepare_n<3>();
    case 4: return prepare_n<4>();
    case 5: return prepare_n<5>();
  }
  return cudaErrorInvalidValue;
}

cudaError_t DG_LAUNCH_NAME(int N, const StageArgs& a, cudaStream_t st) {
  switch (N) {
    case 1: return launch_n<1>(a, st);
    case 2: return launch_n<2>(a, st);
    case 3: return launch_n<3>(a, st);
    case 4: return launch_n<4>(a, st);
    case 5: return launch_n<5>(a, st);
  }
  return cudaErrorInvalidValue;
}
