// stage_kernel.cuh -- the fused SSP-RK stage kernel of the CUDA path (sm_100a, fp64).
//
// One launch = one SSP-RK stage (PAPER.md:128-152 order of operations) over the whole mesh; a thread
// block owns a tile of TX x TY x TZ elements and a THREAD OWNS (A SEGMENT OF) ONE x-LINE of an element:
// SEG consecutive nodes i at fixed (j,k) -- the whole line of N = p+1 nodes, except for p = 3, where a
// line is split into two 2-node segments so that the 64-node hexahedron is exactly one warp and twice
// as many warps are resident.  Consequences of that mapping:
//   * the line is contiguous in the canonical layout X[v][e][n], n = i + N (j + N k): every state
//     access of a thread is a 16-byte vector access (N even) and a warp reads / writes whole 128-byte
//     lines; the neighbours' facing nodal layers in y and z are lines too (16-byte cp.async);
//   * the x-direction volume contraction (Eq. 17) runs in registers (whole-line threads) or from the
//     line's own records; the y and z contractions read the line-mates' records from shared memory
//     with 16-byte loads (natural node order: the nodes of a thread are adjacent);
//   * a cell is at most 32 consecutive lanes of ONE warp, so everything cell-local in the
//     physicality operator (cell mean, min s) is a warp shuffle: no shared memory, no barrier;
//   * SEG independent fp64 instruction streams per thread (con2prim's Newton iteration in lockstep).
// Inputs per node: the stage state U_s and its pressure P_s = P(U_s), recovered by the stage that
// produced U_s (8 B per node; everything else the flux and the wave speeds need follows from (U, P)
// without a square root, physics.cuh dg_derive).  Primitives are never stored.
// Steps:
//   1. own lines and the one-node-deep face layers of the neighbouring elements (GLL nodes: the face
//      interpolation of :132-134 is a gather, reading R1; periodic wrap / outflow copy, R12) -> records
//      in shared memory: U, P and r = 1/(E+P) (v = M r; the fraction sigma = num/den of Eq. 22 is
//      re-derived at the face points);
//   2. interface flux -- HLL (Eq. 21-24, reading R9) or HLLC (ref [34]) -- at every face point of the
//      tile, once each, spread over the block's threads; ghost states at the mesh boundary: outflow
//      copy, reflecting wall or fixed (Dirichlet) state; volume quadrature (Eq. 17) over the diagonal mass matrix, F_d =
//      U v_d + P e_d (Eq. 2) formed on the fly from the records;
//   3. surface lift (Eq. 18).  MODE_RHS stops here and writes R = L(U).  MODE_STAGE continues:
//   4. SSP-RK combine  U_out = a U0 + b (U_s + dt R)   (:147-152, reading R10), dt from device memory;
//   5. physicality-enforcing operator on the cell (Eq. 25-37, :242-252);
//   6. pressure of the new state (con2prim, Eq. 16 for the next stage) and, on the step's last stage,
//      the CFL wave-speed maximum (reading R11): warp shuffle -> one atomicMax per block.
// Algorithmic HBM traffic per node and stage: U_s 40 B + P_s 8 B in, U0 40 B in (a != 0), U_out 40 B +
// P_out 8 B out = 96 / 136 B (mean over SSPRK3: 122.7 B); halo layers are L2 hits.
#pragma once
#ifdef DG_DEBUG_ASSERTS
#include <cstdio>   // device printf of the bounds checks (debug build only)
#endif
#include "physics.cuh"

#define DG_MODE_RHS 0
#define DG_MODE_STAGE 1
#define DG_BC_PERIODIC 0
#define DG_BC_OUTFLOW 1
#define DG_BC_REFLECT 2
#define DG_BC_DIRICHLET 3
#define DG_RS_HLL 0
#define DG_RS_HLLC 1
#define DG_NSLOT 32          // counter / CFL-maximum slots (spread same-address atomics), 128 B apart
#define DG_SLOT_STRIDE 16    // in 8-byte words

typedef unsigned long long dg_ull;

__host__ __device__ constexpr int dg_ipow(int b, int e) { return e <= 0 ? 1 : b * dg_ipow(b, e - 1); }

// elements per thread block along x,y,z for [ndim-1][N-1]
// (3D p=3: 2x2x2 elements = 512 nodes = 8 warps of 2-node threads, two blocks per SM on shared memory)
__host__ __device__ constexpr int dg_tile(int nd, int N, int d) {
  constexpr int t[3][5][3] = {
      {{64, 1, 1}, {64, 1, 1}, {64, 1, 1}, {64, 1, 1}, {64, 1, 1}},
      {{16, 8, 1}, {16, 4, 1}, {10, 4, 1}, {8, 4, 1}, {6, 4, 1}},
      {{8, 4, 4}, {4, 4, 2}, {3, 2, 2}, {2, 2, 2}, {2, 2, 1}}};
  return t[nd - 1][N - 1][d];
}

template <int ND, int N>
struct TileShape {
  static constexpr int NN = dg_ipow(N, ND);          // nodes per element
  static constexpr int NF1 = dg_ipow(N, ND - 1);     // nodes per element face = x-lines per element
  static constexpr int SEG = (N == 4) ? 2 : N;       // nodes per thread (a segment of an x-line)
  static constexpr int NSEG = N / SEG;               // segments per line
  static constexpr int NL = NSEG * NF1;              // threads per element
  static constexpr int TX = dg_tile(ND, N, 0), TY = dg_tile(ND, N, 1), TZ = dg_tile(ND, N, 2);
  static constexpr int NE = TX * TY * TZ;            // elements per tile
  static constexpr int EPW = 32 / NL;                // elements per warp (lanes >= EPW*NL idle)
  static constexpr int NW = (NE + EPW - 1) / EPW;    // warps per block
  static constexpr int NT = 32 * NW;                 // threads per block
  // shared-memory slot of node (i,j,k) of tile element le: le*ES + i + N*j + PK*k (natural order: the
  // 16-byte line loads of a quarter-warp fall into distinct banks or coincide)
  static constexpr int PK = (ND == 3) ? N * N : 0;
  static constexpr int ES = (ND == 1) ? N : ((ND == 2) ? N * N : N * PK);
  static constexpr int NS = (NE * ES + 1) / 2 * 2;   // slots per record row
  __host__ __device__ static constexpr int T(int d) { return d == 0 ? TX : (d == 1 ? TY : TZ); }
  __host__ __device__ static constexpr int SE(int d) { return d == 0 ? 1 : (d == 1 ? TX : TX * TY); }
  __host__ __device__ static constexpr int SS(int d) { return d == 0 ? 1 : (d == 1 ? N : PK); }
  // Slot of the segment h of line (j,k) of tile element le, and of node (i,j,k).  For the 64-node
  // hexahedron (two 16-byte segments per line) the four lines of a k-plane are rotated by k lines and
  // the two segments of a line swapped for odd k: the line loads of the volume terms stay conflict-free,
  // the y- and z-face loads become conflict-free, and the x-face points -- which read nodes of one
  // parity of i only (4-way bank conflicts in the natural order) -- reach the 2-way floor.
  static constexpr bool SWZ = (ND == 3 && N == 4);
  __host__ __device__ static constexpr int seg_slot(int le, int h, int j, int k) {
    return SWZ ? le * ES + 16 * k + 4 * ((j + k) & 3) + 2 * (h ^ (k & 1)) : le * ES + h * SEG + N * j + PK * k;
  }
  __host__ __device__ static constexpr int node_slot(int le, int i, int j, int k) {
    return SWZ ? seg_slot(le, i >> 1, j, k) + (i & 1) : le * ES + i + N * j + PK * k;
  }
  __host__ __device__ static constexpr int FP(int d) { return NE / T(d) * NF1; }   // points per face plane
  __host__ __device__ static constexpr int HOFF(int d) { return d <= 0 ? 0 : HOFF(d - 1) + 2 * FP(d - 1); }
  __host__ __device__ static constexpr int FOFF(int d) {
    return d <= 0 ? 0 : FOFF(d - 1) + (T(d - 1) + 1) * FP(d - 1);
  }
  // interior face planes only (the flux of a boundary plane is kept in its halo slot, see below)
  __host__ __device__ static constexpr int FOFFI(int d) {
    return d <= 0 ? 0 : FOFFI(d - 1) + (T(d - 1) - 1) * FP(d - 1);
  }
  // interface fluxes: direction D holds T(D)+1 face planes of PS(D) doubles, a plane = 5 components of
  // FP(D) points (+ padding: consecutive y-planes of the 64-node hexahedron are shifted by 32 bytes so
  // that the lift's 16-byte loads of the minus and the plus face fall into different banks)
  __host__ __device__ static constexpr int PS(int d) { return 5 * FP(d) + ((SWZ && d == 1) ? 4 : 0); }
  __host__ __device__ static constexpr int FHOFF(int d) {
    return d <= 0 ? 0 : FHOFF(d - 1) + (T(d - 1) + 1) * PS(d - 1);
  }
  static constexpr int NHALO = HOFF(ND);             // halo points of the tile
  static constexpr int NHP = (NHALO + 1) / 2 * 2;    // halo slots per row (even)
  static constexpr int NFACE = FOFF(ND);             // face points of the tile (all directions)
  static constexpr int NFACEI = FOFFI(ND);           // of which between two elements of the tile
  // shared memory, in doubles.  Records X[7][RS]: row = D Mx My Mz E | P | r (conserved state, pressure,
  // r = 1/(E+P): v = M r); a row holds the NS node slots of the tile followed by its NHP halo points
  // (rows 0..5 only), so that a face point addresses either kind of side with the same row stride.
  // Shared-memory bandwidth is a co-equal bound of this kernel, so the records hold only what cannot
  // be re-derived in a few flops.
  static constexpr int NREC = 7;
  static constexpr int RS = NS + NHP;                // row stride
  static constexpr int O_X = 0;
  static constexpr int O_FH = O_X + NREC * RS;       // Fhat  [dir][plane][5][FP]
  static constexpr int O_D = O_FH + (FHOFF(ND) + 1) / 2 * 2;   // (2/h_d) Dhat[i][q] for d = x, y, z
  static constexpr int SMEM_BYTES = (O_D + 3 * 26) * 8;
  static constexpr int BLK_SMEM = (227 * 1024) / (SMEM_BYTES + 1024);
  // (3-node lines: 96 registers / 5 blocks of 128 threads measured 3.7 % faster than 112 / 4 on the 2D p=2
  // shear layer; 80 / 6 spills and is 9 % slower)
  static constexpr int REG_FLOOR = (SEG <= 1) ? 64 : ((SEG >= 6) ? 240 : (SEG == 3 ? 96 : 40 * SEG));   // registers per thread to leave
  static constexpr int BLK_REG = 65536 / (NT * REG_FLOOR);
  static constexpr int MINB = (BLK_SMEM < BLK_REG ? BLK_SMEM : BLK_REG) > 0 ? (BLK_SMEM < BLK_REG ? BLK_SMEM : BLK_REG) : 1;
};

struct StageArgs {
  const double* Us;       // U_s[5][ndof]   stage input state (16-byte aligned if N is even)
  const double* Pin;      // P_s[ndof]      its pressure
  const double* U0;       // U at the start of the step (read only if a != 0); may alias Uout
  double* Uout;           // must not alias Us (neighbouring blocks read their halo from Us)
  double* Pout;           // must not alias Pin
  double* Rout;           // MODE_RHS: R = L(U_s)
  long long ndof;
  int ne[3];
  double a, b;            // Shu-Osher coefficients of this stage
  const double* dt_ptr;   // device
  double f_screen, f_solve, one_m_delta;   // 1-eps_q/2, 1-eps_q, 1-delta_s
  EosPar eos;
  double cw[3];           // (2p+1)/h_d
  dg_ull* amax;           // [DG_NSLOT] ordered-int images of the CFL maximum (atomicMax)
  int do_cfl;
  dg_ull* counters;       // [DG_NSLOT][n_flagged, n_bad_mean, n_c2p_fail, n_tm_fallback]
  double Dx[25];          // (2/h_x) Dhat[i*N+q]
  double Dy[25], Dz[25];
  double w[5];            // GLL weights
  double lift[3];         // (2/h_d) / w_0
  double wsum;            // sum of the tensor weights
  int mode;               // DG_MODE_RHS / DG_MODE_STAGE
  int hoff[3][2], hfix[3][2];   // halo: global-index offset of the facing node (minus, plus side)
  int bcm[3][2];          // at a mesh boundary [axis][end]: 0 ghost = halo value as loaded (periodic wrap /
                          // outflow copy), DG_BC_REFLECT normal momentum reversed, DG_BC_DIRICHLET fixed state
  double bcU[3][2][6];    // Dirichlet ghost state: U (Eq. 4 of the given primitives) and P
  int lby, lbz;           // 3D launch order: tiles are walked in bricks of (all x) x 2^lby x 2^lbz tiles, see
                          // dg_tile_of_block; 0, 0 = plain x-fastest order (grid = tile grid)
};

// Tile (y, z) index of a block.  The hardware starts blocks in blockIdx order, x fastest, then y, then z.
// In that plain order the z-neighbour of a tile runs a whole xy-plane of tiles later (4096 tiles = ~100 MB
// of traffic at 128^3, p = 3: its halo rows have left L2 by then).  Brick order keeps both neighbours
// close: blockIdx.y = ty_local + BY (tz_local + BZ * brick_y), blockIdx.z = brick_z, BY = 2^lby,
// BZ = 2^lbz, so the z-neighbour runs ntx * BY tiles later.  The launch pads the tile grid to whole
// bricks; blocks of the padding return at once.
DG_INL void dg_tile_of_block(const StageArgs& a, int& ty, int& tz) {
  const int by = (int)blockIdx.y;
  ty = (by & ((1 << a.lby) - 1)) | ((by >> (a.lby + a.lbz)) << a.lby);
  tz = ((by >> a.lby) & ((1 << a.lbz) - 1)) + ((int)blockIdx.z << a.lbz);
}

// ---------------------------------------------------------------------------------------------
// line access helpers: N consecutive doubles, 16-byte vectors when N is even (p 16-byte aligned)
// ---------------------------------------------------------------------------------------------
template <int N>
DG_INL void dg_ld_line(const double* p, double x[N]) {
  if (N % 2 == 0) {
#pragma unroll
    for (int m = 0; m < N / 2; ++m) {
      const double2 t = *reinterpret_cast<const double2*>(p + 2 * m);
      x[2 * m] = t.x; x[2 * m + 1] = t.y;
    }
  } else {
#pragma unroll
    for (int m = 0; m < N; ++m) x[m] = p[m];
  }
}
template <int N>
DG_INL void dg_ldg_line(const double* p, double x[N]) {      // read-only global data
  if (N % 2 == 0) {
#pragma unroll
    for (int m = 0; m < N / 2; ++m) {
      const double2 t = __ldg(reinterpret_cast<const double2*>(p + 2 * m));
      x[2 * m] = t.x; x[2 * m + 1] = t.y;
    }
  } else {
#pragma unroll
    for (int m = 0; m < N; ++m) x[m] = __ldg(p + m);
  }
}
template <int N>
DG_INL void dg_st_line(double* p, const double x[N]) {
  if (N % 2 == 0) {
#pragma unroll
    for (int m = 0; m < N / 2; ++m) *reinterpret_cast<double2*>(p + 2 * m) = make_double2(x[2 * m], x[2 * m + 1]);
  } else {
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = x[m];
  }
}
// asynchronous copy global -> shared of a line (LDGSTS): no register is held while in flight
template <int N>
DG_INL void dg_async_line(double* smem_dst, const double* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  if (N % 2 == 0) {
#pragma unroll
    for (int m = 0; m < N / 2; ++m)
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d + 16 * m), "l"(gmem_src + 2 * m) : "memory");
  } else {
#pragma unroll
    for (int m = 0; m < N; ++m)
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d + 8 * m), "l"(gmem_src + m) : "memory");
  }
}
DG_INL void dg_async_copy8(double* smem_dst, const double* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)),
               "l"(gmem_src) : "memory");
}
DG_INL void dg_async_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// ---------------------------------------------------------------------------------------------
// The physicality-enforcing operator (PAPER.md:242-252 steps 1-4) on the cells of one warp.  A
// thread owns SEG consecutive nodes of an x-line of its cell: Uo[0..SEG-1], limited in place; the NL
// threads of a cell are consecutive lanes starting at a multiple of NL.  MUST be called by all 32
// lanes (inactive lanes pass active = false).  This one function serves the fused stage kernel and
// the stand-alone dgrhd_enforce_physicality kernel.
//   wn[m]: tensor GLL weight of node m of the thread.
//   cnt[0], cnt[1] += cells flagged / cells with an inadmissible mean, counted on the cell's first lane.
// Returns the cell's flag; s_out = blend factor (1 if unflagged, 0 for an inadmissible mean, R13d).
// ---------------------------------------------------------------------------------------------
struct LimPar {
  double w[5];
  double wsum, f_screen, f_solve, one_m_delta;
};

template <int NL>
DG_INL double dg_cell_sum(double x, int base) {
  if ((NL & (NL - 1)) == 0) {                      // power of two: butterfly inside the aligned group
#pragma unroll
    for (int o = NL / 2; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
  }
  double acc = 0.0;                                // fixed lane order, the same on every lane
#pragma unroll
  for (int o = 0; o < NL; ++o) acc += __shfl_sync(0xffffffffu, x, min(base + o, 31));
  return acc;
}
template <int NL>
DG_INL double dg_cell_min(double x, int base) {
  if ((NL & (NL - 1)) == 0) {
#pragma unroll
    for (int o = NL / 2; o > 0; o >>= 1) x = fmin(x, __shfl_xor_sync(0xffffffffu, x, o));
    return x;
  }
  double acc = x;
#pragma unroll
  for (int o = 0; o < NL; ++o) acc = fmin(acc, __shfl_sync(0xffffffffu, x, min(base + o, 31)));
  return acc;
}

// the rare part: everything after the screen has found an inadmissible node in the warp
template <int NL, int SEG>
DG_INL bool dg_limiter_cells_slow(double (*Uo)[5], bool active, int lane, unsigned ball,
                                                          const double* wn, const LimPar& lp, int cnt[2],
                                                          double& s_out) {
  const int base = (lane / NL) * NL;
  const unsigned cmask = ((NL >= 32) ? 0xffffffffu : ((1u << NL) - 1u)) << base;
  const bool flagged = active && ((ball & cmask) != 0u);
  double Ub[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) {                   // cell average: thread partial sums, then across lanes
    double part = 0.0;
    if (flagged) {
#pragma unroll
      for (int m = 0; m < SEG; ++m) part = fma(wn[m], Uo[m][v], part);
    }
    Ub[v] = dg_cell_sum<NL>(part, base) / lp.wsum;
  }
  double si = 1.0;
  bool mean_ok = true;
  if (flagged) {
    mean_ok = dg_admissible(Ub, lp.f_solve);      // step 2 (reading R13d)
    if (mean_ok) {
      DgState5 ub;
#pragma unroll
      for (int v = 0; v < 5; ++v) ub.v[v] = Ub[v];
#pragma unroll
      for (int m = 0; m < SEG; ++m) {
        DgState5 ui;
#pragma unroll
        for (int v = 0; v < 5; ++v) ui.v[v] = Uo[m][v];
        double sm_ = dg_limiter_node_s(ub, ui, lp.f_solve);        // step 3
        if (!(sm_ >= 0.0)) sm_ = 0.0;
        si = fmin(si, sm_);
      }
    } else {
      si = 0.0;
    }
  }
  const double smin = dg_cell_min<NL>(si, base);  // step 4: s = min_i s_i
  if (flagged) {
    const double s = lp.one_m_delta * smin;       // R13c
    const double tt = 1.0 - s;
#pragma unroll
    for (int m = 0; m < SEG; ++m) {
#pragma unroll
      for (int v = 0; v < 5; ++v)                 // Eq. 26 from the nearer end (R14)
        Uo[m][v] = (s > 0.5) ? fma(tt, Ub[v] - Uo[m][v], Uo[m][v]) : fma(s, Uo[m][v] - Ub[v], Ub[v]);
    }
    s_out = s;
    if (lane == base) {
      cnt[0] += 1;
      if (!mean_ok) cnt[1] += 1;
    }
  }
  return flagged;
}

template <int NL, int SEG>
DG_INL bool dg_limiter_cells(double (*Uo)[5], bool active, int lane, const double* wn, const LimPar& lp,
                             int cnt[2], double& s_out) {
  s_out = 1.0;
  bool bad = false;
  if (active) {
#pragma unroll
    for (int m = 0; m < SEG; ++m) bad = bad || !dg_admissible(Uo[m], lp.f_screen);   // step 1: screen (R13e)
  }
  const unsigned ball = __ballot_sync(0xffffffffu, bad);
  if (ball == 0u) return false;                   // nothing flagged in this warp (the common case)
  return dg_limiter_cells_slow<NL, SEG>(Uo, active, lane, ball, wn, lp, cnt, s_out);
}

// ---------------------------------------------------------------------------------------------
// HLL flux (reading R9, Eq. 21-24) at one face point from the two sides' U, normal velocity, P and
// sigma = num/den:  F = cL F_L + cR F_R + cU (U_R - U_L),  F_s = U_s v_s + P_s e_D (+ P_s v_s in
// the energy).  D: the face's direction; pF[v * fstride] receives the flux.
// ---------------------------------------------------------------------------------------------
template <int D>
DG_INL void dg_hll_point(const double UL[5], double vL, double PL, double numL, double denL,
                         const double UR[5], double vR, double PR, double numR, double denR,
                         double* pF, int fstride) {
  double nmL, npL, dL, nmR, npR, dR;
  dg_speeds_frac(vL, numL, denL, nmL, npL, dL);
  dg_speeds_frac(vR, numR, denR, nmR, npR, dR);
  // lambda_L = min(nmL/dL, nmR/dR) =: nl/dl, lambda_R = max(npL/dL, npR/dR) =: nr/dr  (Eq. 23-24),
  // compared by cross-multiplication (dL, dR > 0); the HLL weights then need one division:
  //   (cL, cR, cU) = (nr dl, -nl dr, nl nr) / (nr dl - nl dr).
  const bool ml = nmL * dR <= nmR * dL, mr = npL * dR >= npR * dL;
  const double nl = ml ? nmL : nmR, dl = ml ? dL : dR;
  const double nr = mr ? npL : npR, dr = mr ? dL : dR;
  double cL, cR, cU;
  if (nl >= 0.0) { cL = 1.0; cR = 0.0; cU = 0.0; }
  else if (nr <= 0.0) { cL = 0.0; cR = 1.0; cU = 0.0; }
  else {
    const double aa = nr * dl, bb = nl * dr;
    const double q = dg_rcp(aa - bb);
    cL = aa * q; cR = -bb * q; cU = nl * nr * q;
  }
  const double kL = fma(cL, vL, -cU), kR = fma(cR, vR, cU);
  double f[5];
#pragma unroll
  for (int v = 0; v < 4; ++v) f[v] = fma(kL, UL[v], kR * UR[v]);
  f[1 + D] += fma(cL, PL, cR * PR);
  f[4] = fma(cL, UL[1 + D], fma(cR, UR[1 + D], cU * (UR[4] - UL[4])));   // (E + P) v_n = M_n
#pragma unroll
  for (int v = 0; v < 5; ++v) pF[v * fstride] = f[v];
}

// HLLC flux ("HLL and HLLC variants ... Mignone and Bodo [34]"; formulas only cited)
// from the same inputs: lambda_L, lambda_R of Eq. 23-24; HLL state and flux U^hll, F^hll; the contact
// speed lambda* = minus-sign root of  F_E^hll l^2 - (E^hll + F_m^hll) l + m^hll = 0  (m: momentum
// normal to the face), written as 2c / (-b + sqrt(b^2 - 4ac)), which stays finite as F_E^hll -> 0;
// p* = -F_E^hll l* + F_m^hll; the star state of the side the contact has not passed,
//   D* = D (lK - v)/(lK - l*), m_t* = m_t (lK - v)/(lK - l*), m* = (m (lK - v) + p* - p)/(lK - l*),
//   E* = (E (lK - v) + p* l* - p v)/(lK - l*),  and  F = F_K + lK (U*_K - U_K).
template <int D>
DG_INL void dg_hllc_point(const double UL[5], double vL, double PL, double numL, double denL,
                          const double UR[5], double vR, double PR, double numR, double denR,
                          double* pF, int fstride) {
  double nmL, npL, dL, nmR, npR, dR;
  dg_speeds_frac(vL, numL, denL, nmL, npL, dL);
  dg_speeds_frac(vR, numR, denR, nmR, npR, dR);
  const double rdL = dg_rcp(dL), rdR = dg_rcp(dR);
  const double lL = fmin(nmL * rdL, nmR * rdR), lR = fmax(npL * rdL, npR * rdR);   // Eq. 23-24
  constexpr int m = 1 + D;
  double FL[5], FR[5];
#pragma unroll
  for (int v = 0; v < 4; ++v) { FL[v] = UL[v] * vL; FR[v] = UR[v] * vR; }
  FL[m] += PL; FR[m] += PR;
  FL[4] = UL[m]; FR[4] = UR[m];                                     // (E + P) v_n = M_n
  double f[5];
  if (lL >= 0.0) {
#pragma unroll
    for (int v = 0; v < 5; ++v) f[v] = FL[v];
  } else if (lR <= 0.0) {
#pragma unroll
    for (int v = 0; v < 5; ++v) f[v] = FR[v];
  } else {
    const double inv = dg_rcp(lR - lL);
    const double Um = (lR * UR[m] - lL * UL[m] + FL[m] - FR[m]) * inv;
    const double Ue = (lR * UR[4] - lL * UL[4] + FL[4] - FR[4]) * inv;
    const double Fm = (lR * FL[m] - lL * FR[m] + lL * lR * (UR[m] - UL[m])) * inv;
    const double Fe = (lR * FL[4] - lL * FR[4] + lL * lR * (UR[4] - UL[4])) * inv;
    const double b = -(Ue + Fm);
    const double disc = dg_sqrt(fmax(fma(b, b, -4.0 * Fe * Um), 0.0));
    const double ls = 2.0 * Um * dg_rcp(disc - b);
    const double ps = fma(-Fe, ls, Fm);
    const bool left = (ls >= 0.0);
    const double lK = left ? lL : lR, vK = left ? vL : vR, PK = left ? PL : PR;
    const double den = dg_rcp(lK - ls);
    const double w = lK - vK, fac = w * den;
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      const double Uk = left ? UL[v] : UR[v], Fk = left ? FL[v] : FR[v];
      double Us = Uk * fac;
      if (v == m) Us = (Uk * w + ps - PK) * den;
      if (v == 4) Us = (Uk * w + ps * ls - PK * vK) * den;
      f[v] = fma(lK, Us - Uk, Fk);
    }
  }
#pragma unroll
  for (int v = 0; v < 5; ++v) pF[v * fstride] = f[v];
}

// Where the two sides of face point fl of direction D live: slots of the record rows -- a tile node
// (< NS) or a halo point (>= NS: rows U | P only; r is derived at use, each halo point is used by
// exactly one face point) -- and where its flux goes.  Returns false for face points outside a
// ragged tile.
struct FaceSides {
  int sl, sr;        // record slots of the left / right side
  bool hl, hr;       // side is a halo point
  int of, fstride;   // flux destination: offset from the start of shared memory, component stride
};

template <int ND, int N, int D>
DG_INL bool dg_face_sides(int fl, const int teff[3], FaceSides& fs) {
  using TS = TileShape<ND, N>;
  constexpr int A = (D == 0) ? 1 : 0, B = (D == 2) ? 1 : 2;         // transverse axes (ascending)
  constexpr int FPD = TS::FP(D);
  const int p = fl / FPD, fp = fl - p * FPD;
  const int te = fp / TS::NF1, tn = fp - te * TS::NF1;
  const int la = te % TS::T(A), lb = te / TS::T(A);
  const int ca = tn % N, cb = tn / N;
  if (p > teff[D] || la >= teff[A] || lb >= teff[B]) return false;
  const int telem = la * TS::SE(A) + lb * TS::SE(B);
  // node coordinates of the two sides: the transverse ones are (ca, cb); along D the left side is the
  // last node of element p-1, the right side the first node of element p
  int cl[3], cr[3];
  cl[A] = cr[A] = ca; cl[B] = cr[B] = cb; cl[D] = N - 1; cr[D] = 0;
  fs.hl = (p < 1);
  fs.hr = (p >= teff[D]);
  const int hl_slot = TS::NS + TS::HOFF(D) + fp, hr_slot = hl_slot + FPD;
  fs.sl = fs.hl ? hl_slot : TS::node_slot(telem + (p - 1) * TS::SE(D), cl[0], (ND >= 2) ? cl[1] : 0, (ND >= 3) ? cl[2] : 0);
  fs.sr = fs.hr ? hr_slot : TS::node_slot(telem + p * TS::SE(D), cr[0], (ND >= 2) ? cr[1] : 0, (ND >= 3) ? cr[2] : 0);
  DG_ASSERT(fs.sl >= 0 && fs.sl < TS::RS && fs.sr >= 0 && fs.sr < TS::RS);
  DG_ASSERT(TS::HOFF(D) + FPD + fp < TS::NHALO);
  fs.of = TS::O_FH + TS::FHOFF(D) + p * TS::PS(D) + fp;
  fs.fstride = FPD;
  DG_ASSERT(TS::FHOFF(D) + p * TS::PS(D) + 4 * FPD + fp < TS::FHOFF(ND));
  return true;
}

// bmode (block-uniform): what stands behind a halo point that lies outside the mesh (StageArgs::bcm)
template <int ND, int N, int EOS, int D>
DG_INL void dg_load_side(const EosPar& eos, const double* x, bool halo, int bmode, const double* bcU,
                         double U[5], double& vn, double& P, double& num, double& den) {
  constexpr int S = TileShape<ND, N>::RS;
#pragma unroll
  for (int v = 0; v < 5; ++v) U[v] = x[v * S];
  P = x[5 * S];
  double r;
  if (halo) {
    if (bmode == DG_BC_REFLECT) U[1 + D] = -U[1 + D];               // wall
    if (bmode == DG_BC_DIRICHLET) {                                 // fixed state
#pragma unroll
      for (int v = 0; v < 5; ++v) U[v] = bcU[v];
      P = bcU[5];
    }
    r = dg_rcp(U[4] + P);
  } else {
    r = x[6 * S];
  }
  vn = U[1 + D] * r;
  dg_sigma_r<EOS>(eos, U, P, r, num, den);
}

template <int ND, int N, int EOS, int RSOL, int D>
DG_INL void dg_face_point(const StageArgs& a, double* sm, int fl, const int teff[3], int bm0, int bm1) {
  FaceSides fs;
  if (!dg_face_sides<ND, N, D>(fl, teff, fs)) return;
  double UL[5], UR[5], vL, vR, PL, PR, numL, denL, numR, denR;
  dg_load_side<ND, N, EOS, D>(a.eos, sm + fs.sl, fs.hl, bm0, a.bcU[D][0], UL, vL, PL, numL, denL);
  dg_load_side<ND, N, EOS, D>(a.eos, sm + fs.sr, fs.hr, bm1, a.bcU[D][1], UR, vR, PR, numR, denR);
  if (RSOL == DG_RS_HLLC) dg_hllc_point<D>(UL, vL, PL, numL, denL, UR, vR, PR, numR, denR, sm + fs.of, fs.fstride);
  else dg_hll_point<D>(UL, vL, PL, numL, denL, UR, vR, PR, numR, denR, sm + fs.of, fs.fstride);
}

// Volume term of direction D = 1 (y) or 2 (z) for the SEG nodes of this thread, segment h of line (j,k)
// of tile element le (Eq. 17 over the diagonal mass matrix): for each q the segment at index q along D
// -- SEG adjacent slots -- is read with vector loads and F_D = [D v_D, M v_D + P e_D, M_D], v_D = M_D r, is formed on the fly.
// dh: (2/h_D) Dhat[id][q] of this thread's index id along D.
template <int ND, int N, int D>
DG_INL void dg_volume_seg(const double* X, const double* dh, int le, int h, int j, int k, double (*R)[5]) {
  using TS = TileShape<ND, N>;
  constexpr int S = TS::RS, SEG = TS::SEG;
#pragma unroll
  for (int q = 0; q < N; ++q) {
    const double* x = X + ((D == 1) ? TS::seg_slot(le, h, q, k) : TS::seg_slot(le, h, j, q));
    const double c = dh[q];
    double u[4][SEG], Pq[SEG], rq[SEG];
#pragma unroll
    for (int v = 0; v < 4; ++v) dg_ld_line<SEG>(x + v * S, u[v]);
    dg_ld_line<SEG>(x + 5 * S, Pq);
    dg_ld_line<SEG>(x + 6 * S, rq);
#pragma unroll
    for (int m = 0; m < SEG; ++m) {
      const double md = u[1 + D][m];
      const double t = (c * rq[m]) * md;                 // (2/h) Dhat v_D
#pragma unroll
      for (int v = 0; v < 4; ++v) R[m][v] = fma(t, u[v][m], R[m][v]);
      R[m][1 + D] = fma(c, Pq[m], R[m][1 + D]);
      R[m][4] = fma(c, md, R[m][4]);
    }
  }
}

// Volume term of direction x for a thread that owns only a segment of its line: the line's segments
// (SEG adjacent slots each) are read one after the other; dh: rows (2/h_x) Dhat[i0+m][.] of the
// thread's nodes.
template <int ND, int N>
DG_INL void dg_volume_x_seg(const double* X, const double* dh, int le, int j, int k, double (*R)[5]) {
  using TS = TileShape<ND, N>;
  constexpr int S = TS::RS, SEG = TS::SEG, NSEG = TS::NSEG;
#pragma unroll
  for (int g = 0; g < NSEG; ++g) {
    const double* x = X + TS::seg_slot(le, g, j, k);
    double u[4][SEG], Pq[SEG], rq[SEG], c[SEG][SEG];
#pragma unroll
    for (int v = 0; v < 4; ++v) dg_ld_line<SEG>(x + v * S, u[v]);
    dg_ld_line<SEG>(x + 5 * S, Pq);
    dg_ld_line<SEG>(x + 6 * S, rq);
#pragma unroll
    for (int m = 0; m < SEG; ++m) dg_ld_line<SEG>(dh + m * N + g * SEG, c[m]);
#pragma unroll
    for (int q = 0; q < SEG; ++q) {
      const double vx = u[1][q] * rq[q];
#pragma unroll
      for (int m = 0; m < SEG; ++m) {
        const double t = c[m][q] * vx;
#pragma unroll
        for (int v = 0; v < 4; ++v) R[m][v] = fma(t, u[v][q], R[m][v]);
        R[m][1] = fma(c[m][q], Pq[q], R[m][1]);
        R[m][4] = fma(c[m][q], u[1][q], R[m][4]);
      }
    }
  }
}

// Flux of face plane p of direction D at face point fp: offset from the start of shared memory;
// stride: the distance between the flux components.
template <int ND, int N, int D>
DG_INL int dg_flux_off(int p, int teffD, int fp, int& stride) {
  using TS = TileShape<ND, N>;
  stride = TS::FP(D);
  return TS::O_FH + TS::FHOFF(D) + p * TS::PS(D) + fp;
}

// Lift of the interface flux of direction D = 1 or 2 onto the thread's nodes (Eq. 18): the segment
// lies in the element's minus face (id == 0: + c Fhat) or plus face (id == N-1: - c Fhat); for
// N == 1 in both.
template <int ND, int N, int D>
DG_INL void dg_lift_seg(const double* sm, int id, int lcD, int teffD, int fp0, double c, double (*R)[5]) {
  using TS = TileShape<ND, N>;
  constexpr int SEG = TS::SEG;
  if (id == 0 || id == N - 1) {
    const bool plus = (N > 1) && (id == N - 1);
    const double cs = plus ? -c : c;
    int st;
    const double* p = sm + dg_flux_off<ND, N, D>(lcD + (plus ? 1 : 0), teffD, fp0, st);
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      double f[SEG];
      dg_ld_line<SEG>(p + v * st, f);
#pragma unroll
      for (int m = 0; m < SEG; ++m) R[m][v] = fma(cs, f[m], R[m][v]);
    }
    if (N == 1) {                                 // the single node lies in both faces
      const double* p2 = sm + dg_flux_off<ND, N, D>(lcD + 1, teffD, fp0, st);
#pragma unroll
      for (int v = 0; v < 5; ++v) R[0][v] = fma(-c, p2[v * st], R[0][v]);
    }
  }
}

// Halo: the facing nodal layer of the neighbouring elements (GLL nodes: the face interpolation of
// :132-134 is a gather, reading R1) -> halo rows U | P, asynchronously.  One UNIT = UW consecutive face
// points of direction D on the tile's minus (side 0) or plus (side 1) boundary, first point fp; used for
// even N, where the units are dealt to the block's threads in flat order (a warp then writes consecutive
// shared-memory addresses).
// Source: the own boundary node's global index + a.hoff (one element over) + a.hfix where the tile
// touches the mesh boundary (periodic wrap or, for the other conditions, the node itself: reading R12).
template <int ND, int N, int D, int UW>
DG_INL void dg_halo_unit(const StageArgs& a, double* XH, const int org[3], const int teff[3], int side, int fp) {
  using TS = TileShape<ND, N>;
  constexpr int A = (D == 0) ? 1 : 0, B = (D == 2) ? 1 : 2;         // transverse axes (ascending)
  const int te = fp / TS::NF1, tn = fp - te * TS::NF1;
  const int la = te % TS::T(A), lb = te / TS::T(A);
  if (la >= teff[A] || lb >= teff[B]) return;                       // ragged tile
  int lc[3], nc[3];
  lc[A] = la; lc[B] = lb; lc[D] = side ? teff[D] - 1 : 0;
  nc[A] = tn % N; nc[B] = tn / N; nc[D] = side ? N - 1 : 0;
  const int e = (org[0] + lc[0]) + a.ne[0] * ((org[1] + lc[1]) + a.ne[1] * (org[2] + lc[2]));
  const bool edge = side ? (org[D] + teff[D] == a.ne[D]) : (org[D] == 0);
  const int g = e * TS::NN + nc[0] + N * (nc[1] + N * nc[2]) + a.hoff[D][side] + (edge ? a.hfix[D][side] : 0);
  DG_ASSERT(g >= 0 && g + UW <= a.ndof && TS::HOFF(D) + side * TS::FP(D) + fp + UW <= TS::NHALO);
  double* dst = XH + (TS::HOFF(D) + side * TS::FP(D) + fp);
#pragma unroll
  for (int v = 0; v < 6; ++v) {
    const double* src = (v < 5) ? a.Us + v * a.ndof + g : a.Pin + g;
    if (UW == 2) dg_async_line<2>(dst + v * TS::RS, src);
    else dg_async_copy8(dst + v * TS::RS, src);
  }
}


template <int ND, int N, int EOS, int RSOL>
__global__ void __launch_bounds__(TileShape<ND, N>::NT, TileShape<ND, N>::MINB)
dg_stage_kernel(const __grid_constant__ StageArgs a) {
  using TS = TileShape<ND, N>;
  constexpr int NN = TS::NN, NT = TS::NT, NL = TS::NL, RS = TS::RS;
  constexpr int SEG = TS::SEG, NSEG = TS::NSEG;
  extern __shared__ __align__(16) double sm[];
  double* X = sm + TS::O_X;                // records: node slots, then (XH) halo slots, row stride RS
  double* XH = X + TS::NS;
  double* sDx = sm + TS::O_D;
  double* sDy = sDx + 26;
  double* sDz = sDy + 26;

  // tile of this block; element, line (j,k) and segment h of this thread
  int ty = (int)blockIdx.y, tz = (int)blockIdx.z;
  if constexpr (ND == 3) {
    dg_tile_of_block(a, ty, tz);
    if (ty * TS::TY >= a.ne[1] || tz * TS::TZ >= a.ne[2]) return;    // padding of the brick grid
  }
  const int org[3] = {(int)blockIdx.x * TS::TX, ty * TS::TY, tz * TS::TZ};
  const int teff[3] = {min(TS::TX, a.ne[0] - org[0]), min(TS::TY, a.ne[1] - org[1]),
                       min(TS::TZ, a.ne[2] - org[2])};
  const int t = threadIdx.x, lane = t & 31, wrp = t >> 5;
  const int ew = lane / NL, lt = lane - ew * NL;
  const int h = lt % NSEG, ln = lt / NSEG;                           // segment, line index j + N k
  const int i0 = h * SEG;
  const int le = wrp * TS::EPW + ew;
  const int j = (ND >= 2) ? ln % N : 0, k = (ND >= 3) ? ln / N : 0;
  const int lc[3] = {le % TS::TX, (le / TS::TX) % TS::TY, le / (TS::TX * TS::TY)};
  const bool active = (ew < TS::EPW) && (le < TS::NE) && lc[0] < teff[0] && lc[1] < teff[1] && lc[2] < teff[2];
  const int s0 = TS::seg_slot(le, h, j, k);                          // slot of the thread's first node
  int g0 = 0;                                                        // its global index; ndof < 2^31
  if (active) g0 = ((org[0] + lc[0]) + a.ne[0] * ((org[1] + lc[1]) + a.ne[1] * (org[2] + lc[2]))) * NN + N * ln + i0;
  const bool xlo = (h == 0), xhi = (h == NSEG - 1);                  // the segment holds node i = 0 / N-1
  if (t < N * N) {
    if (NSEG > 1) sDx[t] = a.Dx[t];
    if (ND >= 2) sDy[t] = a.Dy[t];
    if (ND >= 3) sDz[t] = a.Dz[t];
  }

  // 1a. own nodes: U_s, P_s requested first (HBM latency overlaps the halo bookkeeping below)
  double Ul[5][SEG], Pl[SEG];
  if (active) {
#pragma unroll
    for (int v = 0; v < 5; ++v) dg_ldg_line<SEG>(a.Us + v * a.ndof + g0, Ul[v]);
    dg_ldg_line<SEG>(a.Pin + g0, Pl);
    if (a.mode == DG_MODE_STAGE && a.a != 0.0) {          // U0 is needed last: warm L2 now
#pragma unroll
      for (int v = 0; v < 5; ++v) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.U0 + v * a.ndof + g0));
    }
  }
  // 1b. halo -> halo rows U | P, asynchronously.  Even N (16-byte units): the units are dealt to the
  //     block's threads in flat order (dg_halo_unit), so a warp writes consecutive shared-memory addresses
  //     and every thread issues the same number of copies (3D p=3: 0.84 fewer wavefronts per node).  Odd N
  //     (8-byte copies): each boundary thread fetches the layer facing its own nodes, which measured
  //     3 % faster on the 2D p=2 shear layer.
  if constexpr (N % 2 == 0) {
    {
      constexpr int UW = 2;                                             // 16-byte units along x-lines
      constexpr int NU0 = 2 * TS::FP(0);
      constexpr int NU1 = (ND >= 2) ? 2 * TS::FP(1) / UW : 0, NU2 = (ND >= 3) ? 2 * TS::FP(2) / UW : 0;
      for (int u = t; u < NU0 + NU1 + NU2; u += NT) {
        if (u < NU0) {
          const int sd = u / TS::FP(0);
          dg_halo_unit<ND, N, 0, 1>(a, XH, org, teff, sd, u - sd * TS::FP(0));
        } else if (ND == 2 || u < NU0 + NU1) {
          if constexpr (ND >= 2) {
            constexpr int H = TS::FP(1) / UW;
            const int w = u - NU0, sd = w / H;
            dg_halo_unit<ND, N, 1, UW>(a, XH, org, teff, sd, (w - sd * H) * UW);
          }
        } else {
          if constexpr (ND >= 3) {
            constexpr int H = TS::FP(2) / UW;
            const int w = u - NU0 - NU1, sd = w / H;
            dg_halo_unit<ND, N, 2, UW>(a, XH, org, teff, sd, (w - sd * H) * UW);
          }
        }
      }
    }
  } else {
    // 1b. halo: the facing nodal layer of the neighbouring elements (a.hoff: one element over; a.hfix:
    //     periodic wrap or, at an outflow boundary, the node itself) -> halo rows U | P, asynchronously
    if (active) {
      {                                                                // x: one point per line and side
        const int fp = ln + TS::NF1 * (lc[1] + TS::TY * lc[2]);
        if (xlo && lc[0] == 0) {
          const int g = g0 + a.hoff[0][0] + ((org[0] == 0) ? a.hfix[0][0] : 0);
          DG_ASSERT(g >= 0 && g < a.ndof && TS::HOFF(0) + fp < TS::NHALO);
          double* dst = XH + (TS::HOFF(0) + fp);
  #pragma unroll
          for (int v = 0; v < 5; ++v) dg_async_copy8(dst + v * RS, a.Us + v * a.ndof + g);
          dg_async_copy8(dst + 5 * RS, a.Pin + g);
        }
        if (xhi && lc[0] == teff[0] - 1) {
          const int g = g0 + (SEG - 1) + a.hoff[0][1] + ((org[0] + teff[0] == a.ne[0]) ? a.hfix[0][1] : 0);
          DG_ASSERT(g >= 0 && g < a.ndof && TS::HOFF(0) + TS::FP(0) + fp < TS::NHALO);
          double* dst = XH + (TS::HOFF(0) + TS::FP(0) + fp);
  #pragma unroll
          for (int v = 0; v < 5; ++v) dg_async_copy8(dst + v * RS, a.Us + v * a.ndof + g);
          dg_async_copy8(dst + 5 * RS, a.Pin + g);
        }
      }
      if constexpr (ND >= 2) {                                         // y: the thread's segment of the line
        const int fp0 = i0 + N * k + TS::NF1 * (lc[0] + TS::TX * lc[2]);
        if (j == 0 && lc[1] == 0) {
          const int g = g0 + a.hoff[1][0] + ((org[1] == 0) ? a.hfix[1][0] : 0);
          DG_ASSERT(g >= 0 && g + SEG <= a.ndof && TS::HOFF(1) + fp0 + SEG <= TS::NHALO);
          double* dst = XH + (TS::HOFF(1) + fp0);
  #pragma unroll
          for (int v = 0; v < 5; ++v) dg_async_line<SEG>(dst + v * RS, a.Us + v * a.ndof + g);
          dg_async_line<SEG>(dst + 5 * RS, a.Pin + g);
        }
        if (j == N - 1 && lc[1] == teff[1] - 1) {
          const int g = g0 + a.hoff[1][1] + ((org[1] + teff[1] == a.ne[1]) ? a.hfix[1][1] : 0);
          DG_ASSERT(g >= 0 && g + SEG <= a.ndof && TS::HOFF(1) + TS::FP(1) + fp0 + SEG <= TS::NHALO);
          double* dst = XH + (TS::HOFF(1) + TS::FP(1) + fp0);
  #pragma unroll
          for (int v = 0; v < 5; ++v) dg_async_line<SEG>(dst + v * RS, a.Us + v * a.ndof + g);
          dg_async_line<SEG>(dst + 5 * RS, a.Pin + g);
        }
      }
      if constexpr (ND >= 3) {                                         // z: the thread's segment of the line
        const int fp0 = i0 + N * j + TS::NF1 * (lc[0] + TS::TX * lc[1]);
        if (k == 0 && lc[2] == 0) {
          const int g = g0 + a.hoff[2][0] + ((org[2] == 0) ? a.hfix[2][0] : 0);
          DG_ASSERT(g >= 0 && g + SEG <= a.ndof && TS::HOFF(2) + fp0 + SEG <= TS::NHALO);
          double* dst = XH + (TS::HOFF(2) + fp0);
  #pragma unroll
          for (int v = 0; v < 5; ++v) dg_async_line<SEG>(dst + v * RS, a.Us + v * a.ndof + g);
          dg_async_line<SEG>(dst + 5 * RS, a.Pin + g);
        }
        if (k == N - 1 && lc[2] == teff[2] - 1) {
          const int g = g0 + a.hoff[2][1] + ((org[2] + teff[2] == a.ne[2]) ? a.hfix[2][1] : 0);
          DG_ASSERT(g >= 0 && g + SEG <= a.ndof && TS::HOFF(2) + TS::FP(2) + fp0 + SEG <= TS::NHALO);
          double* dst = XH + (TS::HOFF(2) + TS::FP(2) + fp0);
  #pragma unroll
          for (int v = 0; v < 5; ++v) dg_async_line<SEG>(dst + v * RS, a.Us + v * a.ndof + g);
          dg_async_line<SEG>(dst + 5 * RS, a.Pin + g);
        }
      }
    }
  }
  // 1c. own nodes -> records
  double R[SEG][5];
#pragma unroll
  for (int m = 0; m < SEG; ++m)
#pragma unroll
    for (int v = 0; v < 5; ++v) R[m][v] = 0.0;
  if (active) {
    double rl[SEG];
#pragma unroll
    for (int m = 0; m < SEG; ++m) rl[m] = dg_rcp(Ul[4][m] + Pl[m]);
    DG_ASSERT(s0 >= 0 && s0 + SEG <= TS::NS);
#pragma unroll
    for (int v = 0; v < 5; ++v) dg_st_line<SEG>(X + v * RS + s0, Ul[v]);
    dg_st_line<SEG>(X + 5 * RS + s0, Pl);
    dg_st_line<SEG>(X + 6 * RS + s0, rl);
    // volume term, x direction, for whole-line threads in registers: R_i += sum_q (2/h_x) Dhat[i][q] F_x(q)
    if (NSEG == 1 && N > 1) {
      double Fx[SEG][5];
#pragma unroll
      for (int m = 0; m < SEG; ++m) {
        const double vx = Ul[1][m] * rl[m];
#pragma unroll
        for (int v = 0; v < 4; ++v) Fx[m][v] = Ul[v][m] * vx;
        Fx[m][1] += Pl[m];
        Fx[m][4] = Ul[1][m];
      }
#pragma unroll
      for (int m = 0; m < SEG; ++m)
#pragma unroll
        for (int q = 0; q < SEG; ++q) {
          const double c = a.Dx[m * N + q];
#pragma unroll
          for (int v = 0; v < 5; ++v) R[m][v] = fma(c, Fx[q][v], R[m][v]);
        }
    }
  }
  dg_async_wait();
  __syncthreads();

  // 2. interface flux at every face point of the tile, once each, spread over all threads
  int bm[3][2];                                     // ghost-state rule where the tile touches the mesh boundary
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    bm[d][0] = (org[d] == 0) ? a.bcm[d][0] : 0;
    bm[d][1] = (org[d] + teff[d] == a.ne[d]) ? a.bcm[d][1] : 0;
  }
  for (int f = t; f < TS::NFACE; f += NT) {
    if (ND == 1 || f < TS::FOFF(1)) dg_face_point<ND, N, EOS, RSOL, 0>(a, sm, f, teff, bm[0][0], bm[0][1]);
    else if (ND == 2 || f < TS::FOFF(2))
      dg_face_point<ND, N, EOS, RSOL, (ND > 1 ? 1 : 0)>(a, sm, f - TS::FOFF(1), teff, bm[ND > 1 ? 1 : 0][0], bm[ND > 1 ? 1 : 0][1]);
    else
      dg_face_point<ND, N, EOS, RSOL, (ND > 2 ? 2 : 0)>(a, sm, f - TS::FOFF(2), teff, bm[ND > 2 ? 2 : 0][0], bm[ND > 2 ? 2 : 0][1]);
  }
  //    volume quadrature: reads the records only, so it needs no barrier here
  if (active && N > 1) {
    if constexpr (NSEG > 1) dg_volume_x_seg<ND, N>(X, sDx + i0 * N, le, j, k, R);
    if constexpr (ND >= 2) dg_volume_seg<ND, N, 1>(X, sDy + j * N, le, h, j, k, R);
    if constexpr (ND >= 3) dg_volume_seg<ND, N, 2>(X, sDz + k * N, le, h, j, k, R);
  }
  // U0 is requested before the barrier: its (L2) latency overlaps the wait and the lift
  double U0r[5][SEG];
  const bool need_u0 = (a.mode == DG_MODE_STAGE) && (a.a != 0.0) && active;
  if (need_u0) {
#pragma unroll
    for (int v = 0; v < 5; ++v) dg_ld_line<SEG>(a.U0 + v * a.ndof + g0, U0r[v]);
  }
  __syncthreads();

  // 3. surface lift
  if (active) {
    {
      const int fp = ln + TS::NF1 * (lc[1] + TS::TY * lc[2]);
      if (xlo) {
        int st;
        const double* pm = sm + dg_flux_off<ND, N, 0>(lc[0], teff[0], fp, st);
#pragma unroll
        for (int v = 0; v < 5; ++v) R[0][v] = fma(a.lift[0], pm[v * st], R[0][v]);
      }
      if (xhi) {
        int st;
        const double* pp = sm + dg_flux_off<ND, N, 0>(lc[0] + 1, teff[0], fp, st);
#pragma unroll
        for (int v = 0; v < 5; ++v) R[SEG - 1][v] = fma(-a.lift[0], pp[v * st], R[SEG - 1][v]);
      }
    }
    if constexpr (ND >= 2)
      dg_lift_seg<ND, N, 1>(sm, j, lc[1], teff[1], i0 + N * k + TS::NF1 * (lc[0] + TS::TX * lc[2]), a.lift[1], R);
    if constexpr (ND >= 3)
      dg_lift_seg<ND, N, 2>(sm, k, lc[2], teff[2], i0 + N * j + TS::NF1 * (lc[0] + TS::TX * lc[1]), a.lift[2], R);
  }
  if (a.mode == DG_MODE_RHS) {
    if (active) {
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        double r[SEG];
#pragma unroll
        for (int m = 0; m < SEG; ++m) r[m] = R[m][v];
        dg_st_line<SEG>(a.Rout + v * a.ndof + g0, r);
      }
    }
    return;
  }

  // 4. SSP-RK combine (Shu-Osher form); U_s comes back from the thread's own records
  const double dt = *a.dt_ptr;
  double Uo[SEG][5];
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    double u[SEG];
    dg_ld_line<SEG>(X + v * RS + (active ? s0 : 0), u);
#pragma unroll
    for (int m = 0; m < SEG; ++m) Uo[m][v] = a.b * fma(dt, R[m][v], u[m]);
  }
  if (need_u0) {
#pragma unroll
    for (int v = 0; v < 5; ++v)
#pragma unroll
      for (int m = 0; m < SEG; ++m) Uo[m][v] = fma(a.a, U0r[v][m], Uo[m][v]);
  }

  // 5. physicality-enforcing operator (cell-local: warp shuffles)
  int cnt[4] = {0, 0, 0, 0};
  bool flagged;
  {
    LimPar lp;
#pragma unroll
    for (int m = 0; m < 5; ++m) lp.w[m] = a.w[m];
    lp.wsum = a.wsum; lp.f_screen = a.f_screen; lp.f_solve = a.f_solve; lp.one_m_delta = a.one_m_delta;
    double wl = 1.0;
    if (ND >= 2) wl *= a.w[j];
    if (ND >= 3) wl *= a.w[k];
    double wn[SEG];
#pragma unroll
    for (int m = 0; m < SEG; ++m) wn[m] = wl * ((NSEG > 1 && h > 0) ? a.w[(SEG + m) % 5] : a.w[m]);
    double s_unused;
    flagged = dg_limiter_cells<NL, SEG>(Uo, active, lane, wn, lp, cnt, s_unused);
  }

  // 6. pressure of the new state (for the next stage), CFL maximum.  Nodes of unflagged cells have
  //    passed the screen (stricter than Eq. 25), so con2prim's own admissibility test is skipped there.
  double speed = 0.0;
  if (active) {
    double Po[SEG], Pg[SEG];
    int st[SEG];
    dg_ld_line<SEG>(X + 5 * RS + s0, Pg);                 // Newton starts from the node's previous pressure
    dg_con2prim_n<EOS, SEG, false>(a.eos, Uo, nullptr, Po, st, &cnt[3], flagged, Pg);
#pragma unroll
    for (int m = 0; m < SEG; ++m) cnt[2] += (st[m] != 0) ? 1 : 0;
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      double u[SEG];
#pragma unroll
      for (int m = 0; m < SEG; ++m) u[m] = Uo[m][v];
      dg_st_line<SEG>(a.Uout + v * a.ndof + g0, u);
    }
    dg_st_line<SEG>(a.Pout + g0, Po);
    if (a.do_cfl) {
#pragma unroll
      for (int m = 0; m < SEG; ++m) {
        const double sp = dg_cfl_speed<EOS, ND>(a.eos, Uo[m], Po[m], a.cw);
        if (sp > 0.0) speed = fmax(speed, sp);            // NaN never wins
      }
    }
  }
  // warp totals -> slotted global counters (rare) and CFL maximum (one atomic per warp): no block barrier
  const int slot = (int)((blockIdx.x + 7u * blockIdx.y + 13u * blockIdx.z + 5u * (unsigned)wrp) % DG_NSLOT) * DG_SLOT_STRIDE;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const unsigned any = __ballot_sync(0xffffffffu, cnt[c] != 0);
    if (any) {
      int x = cnt[c];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
      if (lane == 0) atomicAdd(&a.counters[slot + c], (dg_ull)x);
    }
  }
  if (a.do_cfl) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) speed = fmax(speed, __shfl_xor_sync(0xffffffffu, speed, o));
    if (lane == 0 && speed > 0.0) atomicMax(a.amax + slot, dg_ord(speed));
  }
}
