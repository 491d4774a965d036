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

// log2 of the brick edge in tiles along y and z.  Measured at 128^3, p = 3 (profiles/r3_brick_order.md): 4 x 4
// tiles reads least from DRAM (plain order 108.6 / 148.9 / 148.7 B per DOF in the three stages, 4 x 4 bricks
// 101.0 / 143.9 / 141.8, 8 x 8 and 16 x 16 in between); the launch time does not move (the kernel is bound by
// instruction issue, not by DRAM).
constexpr int DG_BRICK_LOG2 = 2;

template <int N>
static cudaError_t launch_n(const StageArgs& a, cudaStream_t st) {
  using TS = TileShape<DG_INST_ND, N>;
  const long long ntx = (a.ne[0] + TS::TX - 1) / TS::TX, nty = (a.ne[1] + TS::TY - 1) / TS::TY,
                  ntz = (a.ne[2] + TS::TZ - 1) / TS::TZ;
  if (ntx <= 0 || nty <= 0 || ntz <= 0 || ntx > 2147483647LL || nty > 65535 || ntz > 65535)
    return cudaErrorInvalidConfiguration;
  long long gy = nty, gz = ntz;
  if (DG_INST_ND == 3) {
    // brick order (dg_tile_of_block): the largest power-of-two brick edge <= the target whose padding
    // adds at most 1/8 to the tile count of that axis; the y extent of the grid holds BZ y-columns
    StageArgs b = a;
    int lby = 0, lbz = 0;
    for (int l = DG_BRICK_LOG2; l > 0 && !lby; --l) if (((nty + (1 << l) - 1) >> l << l) * 8 <= nty * 9) lby = l;
    for (int l = DG_BRICK_LOG2; l > 0 && !lbz; --l) if (((ntz + (1 << l) - 1) >> l << l) * 8 <= ntz * 9) lbz = l;
    const long long py = (nty + (1 << lby) - 1) >> lby << lby;
    if ((py << lbz) > 65535) lbz = 0;
    b.lby = lby;
    b.lbz = lbz;
    gy = py << lbz;
    gz = (ntz + (1 << lbz) - 1) >> lbz;
    dg_stage_kernel<DG_INST_ND, N, DG_INST_EOS, DG_INST_RS>
        <<<dim3((unsigned)ntx, (unsigned)gy, (unsigned)gz), TS::NT, TS::SMEM_BYTES, st>>>(b);
    return cudaGetLastError();
  }
  dg_stage_kernel<DG_INST_ND, N, DG_INST_EOS, DG_INST_RS>
      <<<dim3((unsigned)ntx, (unsigned)gy, (unsigned)gz), TS::NT, TS::SMEM_BYTES, st>>>(a);
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
