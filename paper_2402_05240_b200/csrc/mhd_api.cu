// mhd_api.cu -- C ABI (include/mhd.h) of the B200 VL+CT ideal-MHD step: context, memory
// carving, launch sequence of one step.  Pure CUDA runtime; no torch types.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <cuda_runtime.h>

#include "../../include/mhd.h"
#include "mhd_kernels.cuh"
#include "mhd_stage.cuh"
#include "mhd_ctupdate.cuh"
#include "mhd_small.cuh"

using namespace mhd;

namespace {

const int kMaxProf = 32;

struct Context {
  bool inited = false;
  bool owns_memory = false;
  void *base = nullptr;
  size_t bytes = 0;
  Geo g;
  State8 U, Uh;
  Flux21 F;
  Edge3 E;   // CT edge fields
  Edge3 Er;  // cell-centred reference field, Eq. 18
  Edge3 Bnext;  // face arrays that receive B^{n+1}; swapped with U's after every step
  double *scratch = nullptr;  // staging of the host set/get calls (never a result array)
  size_t guard = 0;           // bytes of the guard band on either side of every array (MHD_GUARD=1), else 0
  Scalars *sc = nullptr;
  cudaStream_t stream = 0;
  long long launches = 0;
  bool rate_valid = false;  // sc->rate_bits holds the CFL rate of the current state
  // CUDA graph of two consecutive {dt; step} passes (after two steps the B ping-pong pointers are
  // back where they were, so the captured arguments stay valid); used by mhd_advance on small grids
  cudaGraphExec_t graph[2] = {nullptr, nullptr};  // one per orientation of the B ping-pong
  double graph_cfl[2] = {0.0, 0.0};
  long long graph_launches = 0;
  int num_sms = 148;
  int stage_ty = MHD_STAGE_TY;  // rows per block of the fused predictor stage (0 = three kernels)
  // launch-bound grids: the whole of mhd_advance as one cooperative kernel (mhd_small.cuh).
  // 0 = mhd_advance on grids of at most MHD_SMALL_MAX_CELLS cells; 1 = mhd_step too, any size (MHD_SMALL=1
  // at mhd_init: parity tests); -1 = never (MHD_SMALL=0)
  int small_mode = 0;
  bool coop = false;
  bool ct_fused = false;        // corrector CT + face update + CFL as one kernel (MHD_CT_FUSED=1; 0.81 ms against 0.36 + 0.43)
  int parity = 0;  // flips with every step (which set of face arrays holds B^n)
  // per-launch event timing (mhd_step_profile)
  int prof_n = -1;  // -1 = off, else number of launches recorded so far
  int prof_cap = 0; // launches the two arrays below can take (they belong to the profiling call in progress)
  cudaEvent_t *prof_ev = nullptr;
  const char **prof_name = nullptr;
};

Context C;
char g_err[512] = "no error";
int run_small(int n_steps, double cfl, double dt_fixed);

int fail(int code, const char *msg) {
  snprintf(g_err, sizeof(g_err), "%s", msg);
  return code;
}

int cuda_fail(cudaError_t e, const char *where) {
  snprintf(g_err, sizeof(g_err), "CUDA error at %s: %s", where, cudaGetErrorString(e));
  return MHD_ERR_CUDA;
}

#define CU(call)                                          \
  do {                                                    \
    cudaError_t e_ = (call);                              \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);   \
  } while (0)

#define LAUNCH_CHECK(name)                                          \
  do {                                                              \
    C.launches++;                                                   \
    cudaError_t e_ = cudaGetLastError();                            \
    if (e_ != cudaSuccess) return cuda_fail(e_, name);              \
    if (C.prof_n >= 0 && C.prof_n < C.prof_cap) {                   \
      C.prof_name[C.prof_n] = name;                                 \
      cudaEventRecord(C.prof_ev[++C.prof_n], C.stream);             \
    }                                                               \
  } while (0)

inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

bool make_geo(Geo &g, int nx, int ny, int nz, double gamma, int recon) {
  if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || recon < 0 || recon > 4) return false;
  g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
  g.ng = 3 + recon_radius(recon);  // stencil radius: PCM 0, PLMC/PLMP 1, PPMC/PPMP 2
  g.ox = round_up(g.ng, 4);
  g.N[0] = round_up(g.ox + nx + g.ng, 8);
  g.N[1] = ny + 2 * g.ng;
  g.N[2] = nz + 2 * g.ng;
  g.s[0] = 1; g.s[1] = g.N[0]; g.s[2] = (long long)g.N[0] * g.N[1];
  g.ntot = g.s[2] * g.N[2];
  for (int a = 0; a < 3; a++) { g.d[a] = 1.0 / g.n[a]; g.id[a] = (double)g.n[a]; g.bc[a] = MHD_BC_PERIODIC; }
  g.gamma = gamma;
  g.gm1inv = 1.0 / (gamma - 1.0);
  g.recon = recon;
  return true;
}

const int kNumArrays = 2 * NFIELD + 21 + 3 + 3 + 3 + 1;  // U, half state, fluxes, edge fields, reference field, B^{n+1}, scratch

size_t array_bytes(const Geo &g) { return ((size_t)g.ntot * sizeof(double) + 255) / 256 * 256; }

// Debug layout (MHD_GUARD=1 in the environment of mhd_workspace_bytes / mhd_init): every array sits between
// two guard bands of four z-planes filled with a NaN pattern, and the arrays themselves start as that
// pattern instead of zero.  A write outside an array lands in a guard band (mhd_debug_guard_errors counts
// the damaged words), a read outside it or of a never-written element yields NaN, which surfaces in the
// parity tests if it reaches a result.  compute-sanitizer is closed on this GPU pool; this is the check
// the library carries itself.
const unsigned long long kGuardPattern = 0x7ff8dead0badf00dull;
size_t guard_bytes(const Geo &g) {
  const char *e = getenv("MHD_GUARD");
  if (!e || !atoi(e)) return 0;
  return ((size_t)4 * g.s[2] * sizeof(double) + 255) / 256 * 256;
}

size_t total_bytes(const Geo &g) { return (array_bytes(g) + 2 * guard_bytes(g)) * kNumArrays + 256; }

__global__ void k_fill_pattern(unsigned long long *p, size_t n, unsigned long long v) {
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) p[t] = v;
}
// words of the guard bands (slots of `slot` words: guard | array | guard) that no longer hold the pattern
__global__ void k_count_guard_damage(const unsigned long long *p, size_t slot, size_t guard, int nslots,
                                     unsigned long long v, unsigned long long *count) {
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < (size_t)nslots * 2 * guard;
       t += (size_t)gridDim.x * blockDim.x) {
    const size_t s_ = t / (2 * guard), w = t % (2 * guard);
    const size_t off = s_ * slot + (w < guard ? w : slot - 2 * guard + w);
    if (p[off] != v) atomicAdd(count, 1ull);
  }
}

dim3 grid1(long long n, int block) { return dim3((unsigned)((n + block - 1) / block)); }

void extents(int f, const Geo &g, int &ex, int &ey, int &ez) {
  ex = g.n[0] + (f == F_BX); ey = g.n[1] + (f == F_BY); ez = g.n[2] + (f == F_BZ);
}

int fill_ghosts(State8 &U) {
  const Geo &g = C.g;
  const int L0 = g.n[0] + 2 * g.ng, L1 = g.n[1] + 2 * g.ng;
  int B = round_up(L0, 32);                  // one thread per x index of a row (grid rows are short)
  if (B > 1024) B = 1024;
  if (B < 64) B = 64;
  const int per = B / (2 * g.ng);            // grid rows per block in the x-column part
  const long long rows = (long long)L1 * 2 * g.ng + 2LL * g.ng * g.n[2] + ((long long)g.n[1] * g.n[2] + per - 1) / per;
  // grid.y <= 65535 holds far beyond what fits in 180 GB (640^3: 15 k rows; 1024^3: 25 k)
  const long long brows = (rows + MHD_GHOST_RPB - 1) / MHD_GHOST_RPB;
  if (brows > 65535) return fail(MHD_ERR_ARG, "grid too large for the ghost-fill launch");
  k_fill_ghosts<<<dim3((L0 + B - 1) / B, (unsigned)brows, NFIELD), B, 0, C.stream>>>(U, g);
  LAUNCH_CHECK("k_fill_ghosts");
  return MHD_OK;
}

Box make_box(int l0, int h0, int l1, int h1, int l2, int h2) {
  Box b;
  b.lo[0] = l0; b.hi[0] = h0; b.lo[1] = l1; b.hi[1] = h1; b.lo[2] = l2; b.hi[2] = h2;
  return b;
}

// Faces per thread of a marching sweep.  A chunk costs its faces plus `extra` iterations (the cell it
// reconstructs without solving a face, the start-up loads; the z sweep also solves one face of the next
// chunk), and the grid should fill the SMs' block slots in whole waves: with few waves (<= 128^3) the
// quantisation decides, with many (>= 256^3) the start-up share does and J ~ 32 is the measured optimum.
#ifndef MHD_MARCH_J
#define MHD_MARCH_J 32
#endif

int march_chunk(int nfaces, long long blocks_per_chunk, int extra, int blocks_per_sm) {
  const double slots = (double)C.num_sms * blocks_per_sm;
  const int n32 = (nfaces + MHD_MARCH_J - 1) / MHD_MARCH_J;
  if ((double)(blocks_per_chunk * n32) > 6.0 * slots) {   // many waves: even chunks of about MHD_MARCH_J
    const int nch = (nfaces + MHD_MARCH_J / 2) / MHD_MARCH_J;   // (0 for a thin slab: one chunk)
    return nch < 1 ? nfaces : (nfaces + nch - 1) / nch;
  }
  int best = nfaces;
  double best_cost = -1.0;
  for (int J = nfaces < 4 ? nfaces : 4; J <= nfaces && J <= 2 * MHD_MARCH_J; J++) {
    const int nch = (nfaces + J - 1) / J;
    if ((nfaces + nch - 1) / nch != J) continue;   // even chunks only
    const double waves = (double)(blocks_per_chunk * nch) / slots;
    const double rounds = (waves <= 4.0) ? ceil(waves) : waves + 0.5;
    const double cost = rounds * (J + extra);
    if (best_cost < 0.0 || cost <= best_cost) { best_cost = cost; best = J; }
  }
  return best;
}

template <int RC>
int launch_corrector_fluxes() {
  const Geo &g = C.g;
  // the 5-cell sweeps keep their window in dynamic shared memory (opt-in above 48 KB for the z sweep)
  const size_t wsm = (recon_radius(RC) == 2) ? (size_t)MHD_WSM_BYTES : 0;  // opted in at mhd_init
  const int n0 = g.n[0], n1 = g.n[1], n2 = g.n[2];
  // faces 0..n along the sweep, transverse -1..n (what CT and the final update need)
  {
    Box fb = make_box(0, n0, -1, n1, -1, n2);
    int nwx = (n0 + 1 + 30) / 31;  // warps per pencil: 31 faces each, faces 0..n0
    long long nw = (long long)nwx * (n1 + 2) * (n2 + 2);
    k_flux_x<RC><<<grid1(nw, 4), 128, 0, C.stream>>>(C.Uh, C.F, g, fb, nwx);
    LAUNCH_CHECK("k_flux_x");
  }
  {
    Box fb = make_box(-1, n0, 0, n1, -1, n2);
    long long nt = (long long)(n0 + 2) * (n2 + 2);
    const int J = march_chunk(n1 + 1, grid1(nt, 128).x, 2, recon_radius(RC) == 2 ? MHD_MINB_FM_PPM : MHD_MINB_FM);
    dim3 grid(grid1(nt, 128).x, (n1 + 1 + J - 1) / J);
    k_flux_march<1, RC, false><<<grid, 128, wsm, C.stream>>>(C.Uh, C.F, g, fb, J, C.U, C.sc);
    LAUNCH_CHECK("k_flux_march<1>");
  }
  {
    Box fb = make_box(-1, n0, -1, n1, 0, n2);
    long long nt = (long long)(n0 + 2) * (n1 + 2);
    const int J = march_chunk(n2 + 1, grid1(nt, 128).x, 3, recon_radius(RC) == 2 ? MHD_MINB_FMZ_PPM : MHD_MINB_FMZ);
    dim3 grid(grid1(nt, 128).x, (n2 + 1 + J - 1) / J);
    k_flux_march<2, RC, true><<<grid, 128, wsm, C.stream>>>(C.Uh, C.F, g, fb, J, C.U, C.sc);
    LAUNCH_CHECK("k_flux_march<2>+update");
  }
  return MHD_OK;
}

// One VL+CT step with the dt held in C.sc->dt.
// Steps 2-5 (PCM + HLLD on cells [-2-r, n+r+1], CT on indices [-1-r, n+r+1], half update of
// cells [-1-r, n+r]).  MHD_STAGE_TY = 0 runs them as three kernels through the flux arrays,
// otherwise as the single fused kernel of mhd_stage.cuh with TY rows per block.
template <int TY>
int launch_stage_kernel(const Box &hb) {
  const Geo &g = C.g;
  const int ntx = (hb.hi[0] - hb.lo[0] + 2 + 29) / 30, nty = (hb.hi[1] - hb.lo[1] + 2 + TY - 3) / (TY - 2);
  const int nz = hb.hi[2] - hb.lo[2] + 1;
  const long long tiles = (long long)ntx * nty;
  const long long slots = (long long)C.num_sms * (TY <= 8 ? 2 : 1);
  // z is cut into chunks so that the tiles fill the SMs in whole waves; every chunk pays two extra planes
  int best = 1;
  long long best_cost = -1;
  for (int c = 1; c <= nz && c <= 64; c++) {
    long long cost = ((tiles * c + slots - 1) / slots) * ((nz + c - 1) / c + 2);
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = c; }
  }
  const int lz = (nz + best - 1) / best;
  const size_t smem = (size_t)MHD_STAGE_COLS * 32 * TY * sizeof(double);
  k_predictor_stage<TY><<<dim3((unsigned)tiles, best), 32 * TY, smem, C.stream>>>(C.U, C.Uh, C.Er, g, hb, C.sc, ntx, lz);
  LAUNCH_CHECK("k_predictor_stage");
  return MHD_OK;
}

int launch_predictor_stage() {
  const Geo &g = C.g;
  const int r = recon_radius(g.recon);
  Box hb;
  for (int a = 0; a < 3; a++) { hb.lo[a] = -1 - r; hb.hi[a] = g.n[a] + r; }
  if (C.stage_ty != 0) return launch_stage_kernel<MHD_STAGE_TY>(hb);
  Box pb;
  for (int a = 0; a < 3; a++) { pb.lo[a] = -2 - r; pb.hi[a] = g.n[a] + r + 1; }
  {
    long long plane = (long long)(pb.hi[0] - pb.lo[0] + 1) * (pb.hi[1] - pb.lo[1] + 1);
    dim3 grid(grid1(plane, 128).x, pb.hi[2] - pb.lo[2] + 1);
    k_predictor_flux<<<grid, 128, 0, C.stream>>>(C.U, C.F, C.Er, g, pb);
    LAUNCH_CHECK("k_predictor_flux");
  }
  {
    Box eb = hb;
    for (int a = 0; a < 3; a++) eb.hi[a] += 1;
    long long plane = (long long)(eb.hi[0] - eb.lo[0] + 1) * (eb.hi[1] - eb.lo[1] + 1);
    dim3 grid(grid1(plane, 256).x, eb.hi[2] - eb.lo[2] + 1);
    k_ct<<<grid, 256, 0, C.stream>>>(C.F, C.Er, C.E, g, eb);
    LAUNCH_CHECK("k_ct(predictor)");
    dim3 gridu(grid1(plane, 256).x, eb.hi[2] - eb.lo[2] + 1);
    k_update<true><<<gridu, 256, 0, C.stream>>>(C.U, C.Uh, C.F, C.E, C.Er, g, hb, C.sc, 0.5);
    LAUNCH_CHECK("k_update(half)");
  }
  return MHD_OK;
}

int step_kernels() {
  const Geo &g = C.g;
  const int r = recon_radius(g.recon);
  // One boundary update per step.  k_predictor_stage, the only reader of U^n outside the
  // active cells, applies the boundary map to its own loads (mhd_stage.cuh): the ghost layers are then
  // filled only by mhd_set_state; the three-kernel predictor reads filled layers.
  int rc = MHD_OK;
  if (C.stage_ty == 0) rc = fill_ghosts(C.U);
  if (rc) return rc;
  rc = launch_predictor_stage();
  if (rc) return rc;
  // Steps 6-7: reconstruction + HLLD from U^{n+1/2}
  switch (g.recon) {
    case 0: rc = launch_corrector_fluxes<0>(); break;
    case 1: rc = launch_corrector_fluxes<1>(); break;
    case 2: rc = launch_corrector_fluxes<2>(); break;
    case 3: rc = launch_corrector_fluxes<3>(); break;
    default: rc = launch_corrector_fluxes<4>(); break;
  }
  if (rc) return rc;
  // Step 8 (G12): CT with the corrector fluxes and the half-step reference state, indices [0, n];
  // Step 9: faces 0..n of B^{n+1} (the hydro variables were updated by the z sweep); CFL rate of U^{n+1}.
  // One kernel (mhd_ctupdate.cuh); MHD_CT_FUSED=0 at mhd_init selects the two separate kernels.
  // B^{n+1} goes to a second set of face arrays which then become the state's (pointer swap): a thread
  // reads B^n on faces owned by other threads.
  {
    State8 out = C.U;
    for (int a = 0; a < 3; a++) out.f[F_BX + a] = C.Bnext.f[a];
    if (C.ct_fused) {
      constexpr int TY = MHD_CTU_TY;
      const int ntx = (g.n[0] + 1 + 30) / 31, nty = (g.n[1] + 1 + TY - 2) / (TY - 1);
      const long long tiles = (long long)ntx * nty;
      const long long slots = (long long)C.num_sms * MHD_MINB_CTU;
      // z is cut into chunks so that the tiles fill the SMs in whole waves; every chunk pays one extra plane
      int best = 1;
      long long best_cost = -1;
      const int nz = g.n[2];
      for (int c = 1; c <= nz && c <= 64; c++) {
        long long cost = ((tiles * c + slots - 1) / slots) * ((nz + c - 1) / c + 1);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = c; }
      }
      const int lz = (nz + best - 1) / best;
      k_ct_update<TY><<<dim3((unsigned)tiles, (nz + lz - 1) / lz), 32 * TY, CtuTile<TY>::BYTES, C.stream>>>(C.U, C.Bnext, C.F, C.Er, g, C.sc, ntx, lz);
      LAUNCH_CHECK("k_ct_update+cfl");
    } else {
      Box ab, eb;
      for (int a = 0; a < 3; a++) { ab.lo[a] = 0; ab.hi[a] = g.n[a] - 1; eb.lo[a] = 0; eb.hi[a] = g.n[a]; }
      long long plane = (long long)(g.n[0] + 1) * (g.n[1] + 1);
      dim3 grid(grid1(plane, 256).x, g.n[2] + 1);
      k_ct<<<grid, 256, 0, C.stream>>>(C.F, C.Er, C.E, g, eb);
      LAUNCH_CHECK("k_ct(corrector)");
      k_update<false><<<grid, 256, 0, C.stream>>>(C.U, out, C.F, C.E, C.Er, g, ab, C.sc, 1.0);
      LAUNCH_CHECK("k_update(B)+cfl");
    }
    for (int a = 0; a < 3; a++) { C.Bnext.f[a] = C.U.f[F_BX + a]; C.U.f[F_BX + a] = out.f[F_BX + a]; }
    C.parity ^= 1;
    C.rate_valid = true;
  }
  return MHD_OK;
}

void drop_graph() {
  for (int p = 0; p < 2; p++) {
    if (C.graph[p]) cudaGraphExecDestroy(C.graph[p]);
    C.graph[p] = nullptr;
  }
}

int step_kernels();

// Capture {k_finish_dt; step} x 2 on the library stream.  Launch-latency matters only for grids that
// fit in L2 (32^3, 256x16x16: ~12 launches of a few microseconds each per step).
int build_graph(double cfl) {
  const int p = C.parity;
  if (C.graph[p]) cudaGraphExecDestroy(C.graph[p]);
  C.graph[p] = nullptr;
  cudaGraph_t gr = nullptr;
  long long l0 = C.launches;
  CU(cudaStreamBeginCapture(C.stream, cudaStreamCaptureModeRelaxed));
  int rc = MHD_OK;
  for (int s = 0; s < 2 && !rc; s++) {
    k_finish_dt<<<1, 1, 0, C.stream>>>(C.sc, cfl);
    C.launches++;
    rc = step_kernels();
  }
  cudaError_t e = cudaStreamEndCapture(C.stream, &gr);
  C.graph_launches = C.launches - l0;
  C.launches = l0;
  if (rc) { if (gr) cudaGraphDestroy(gr); return rc; }
  if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
  e = cudaGraphInstantiate(&C.graph[p], gr, 0);
  cudaGraphDestroy(gr);
  if (e != cudaSuccess) { C.graph[p] = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
  C.graph_cfl[p] = cfl;
  return MHD_OK;
}

// CFL rate of the current state into sc->rate_bits, unless the last full update left it there
int ensure_rate() {
  if (C.rate_valid) return MHD_OK;
  const Geo &g = C.g;
  k_reset_rate<<<1, 1, 0, C.stream>>>(C.sc);
  LAUNCH_CHECK("k_reset_rate");
  long long plane = (long long)g.n[0] * g.n[1];
  dim3 grid(grid1(plane, 256).x, g.n[2]);
  k_cfl<<<grid, 256, 0, C.stream>>>(C.U, g, C.sc);
  LAUNCH_CHECK("k_cfl");
  C.rate_valid = true;
  return MHD_OK;
}

// the 5-cell sweeps use more than 48 KB of shared memory per block (window + update operands)
template <int RC>
int opt_in_shared_memory() {
  CU(cudaFuncSetAttribute(k_flux_march<1, RC, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, MHD_WSM_BYTES));
  CU(cudaFuncSetAttribute(k_flux_march<2, RC, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, MHD_WSM_BYTES));
  return MHD_OK;
}

int init_common(int nx, int ny, int nz, double gamma, int recon, void *ws, size_t ws_bytes) {
  mhd_finalize();
  if (recon == MHD_RECON_PPMC || recon == MHD_RECON_PPMP) {
    int rc = (recon == MHD_RECON_PPMC) ? opt_in_shared_memory<2>() : opt_in_shared_memory<4>();
    if (rc) return rc;
  }
  Geo g;
  if (!make_geo(g, nx, ny, nz, gamma, recon)) return fail(MHD_ERR_ARG, "mhd_init: bad argument");
  {
    const int cols = MHD_STAGE_COLS * 32 * (int)sizeof(double);
    CU(cudaFuncSetAttribute(k_predictor_stage<MHD_STAGE_TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, cols * MHD_STAGE_TY));
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    C.num_sms = sms > 0 ? sms : 148;
    CU(cudaFuncSetAttribute(k_ct_update<MHD_CTU_TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CtuTile<MHD_CTU_TY>::BYTES));
    const char *e = getenv("MHD_STAGE_TY");
    if (e) C.stage_ty = atoi(e);
    e = getenv("MHD_SMALL");
    if (e) C.small_mode = atoi(e) ? 1 : -1;
    int coop = 0;
    CU(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    C.coop = coop != 0;
    e = getenv("MHD_CT_FUSED");
    if (e) C.ct_fused = atoi(e) != 0;
  }
  size_t need = total_bytes(g);
  if (ws) {
    if (ws_bytes < need || ((size_t)ws & 255)) return fail(MHD_ERR_NOMEM, "workspace too small or misaligned");
    C.base = ws; C.owns_memory = false;
  } else {
    cudaError_t e = cudaMalloc(&C.base, need);
    if (e != cudaSuccess) { cudaGetLastError(); C.base = nullptr; return fail(MHD_ERR_NOMEM, "cudaMalloc failed"); }
    C.owns_memory = true;
  }
  C.bytes = need;
  C.g = g;
  char *p = (char *)C.base;
  const size_t gb = guard_bytes(g);
  const size_t ab = array_bytes(g) + 2 * gb;   // one slot: guard | array | guard
  C.guard = gb;
  C.sc = (Scalars *)p; p += 256;
  p += gb;                                     // array pointers point past the leading guard
  for (int f = 0; f < NFIELD; f++) { C.U.f[f] = (double *)p; p += ab; }
  for (int f = 0; f < NFIELD; f++) { C.Uh.f[f] = (double *)p; p += ab; }
  for (int a = 0; a < 3; a++)
    for (int c = 0; c < 7; c++) { C.F.f[a][c] = (double *)p; p += ab; }
  for (int a = 0; a < 3; a++) { C.E.f[a] = (double *)p; p += ab; }
  for (int a = 0; a < 3; a++) { C.Er.f[a] = (double *)p; p += ab; }
  for (int a = 0; a < 3; a++) { C.Bnext.f[a] = (double *)p; p += ab; }
  C.scratch = (double *)p; p += ab;
  C.launches = 0;
  C.rate_valid = false;
  C.inited = true;
  cudaError_t e = cudaMemsetAsync(C.base, 0, need, C.stream);
  if (e != cudaSuccess) { mhd_finalize(); return cuda_fail(e, "cudaMemsetAsync"); }
  if (gb) {   // guards AND arrays start as the NaN pattern (the scalars stay zero)
    k_fill_pattern<<<1024, 256, 0, C.stream>>>((unsigned long long *)((char *)C.base + 256), (need - 256) / 8, kGuardPattern);
    LAUNCH_CHECK("k_fill_pattern");
  }
  k_reset_rate<<<1, 1, 0, C.stream>>>(C.sc);
  LAUNCH_CHECK("k_reset_rate");
  return MHD_OK;
}

int set_state_from(const double *const src[NFIELD], bool host) {
  const Geo &g = C.g;
  for (int f = 0; f < NFIELD; f++)
    if (!src[f]) return fail(MHD_ERR_ARG, "mhd_set_state: null pointer");
  for (int f = 0; f < NFIELD; f++) {
    int ex, ey, ez;
    extents(f, g, ex, ey, ez);
    long long cnt = (long long)ex * ey * ez;
    const double *dsrc = src[f];
    if (host) {  // staged through the scratch array; stream order keeps the fields apart
      double *stage = C.scratch;
      CU(cudaMemcpyAsync(stage, src[f], cnt * sizeof(double), cudaMemcpyHostToDevice, C.stream));
      dsrc = stage;
    }
    k_unpack<<<grid1(cnt, 256), 256, 0, C.stream>>>(C.U.f[f], dsrc, g, ex, ey, ez);
    LAUNCH_CHECK("k_unpack");
  }
  C.rate_valid = false;
  return fill_ghosts(C.U);
}

int get_state_to(State8 &S, double *const dst[NFIELD], bool host) {
  const Geo &g = C.g;
  for (int f = 0; f < NFIELD; f++) {
    if (!dst[f]) continue;
    int ex, ey, ez;
    extents(f, g, ex, ey, ez);
    long long cnt = (long long)ex * ey * ez;
    double *ddst = host ? C.scratch : dst[f];
    k_pack<<<grid1(cnt, 256), 256, 0, C.stream>>>(ddst, S.f[f], g, ex, ey, ez);
    LAUNCH_CHECK("k_pack");
    if (host) CU(cudaMemcpyAsync(dst[f], ddst, cnt * sizeof(double), cudaMemcpyDeviceToHost, C.stream));
  }
  return MHD_OK;
}

#ifndef MHD_SMALL_MAX_CELLS
#define MHD_SMALL_MAX_CELLS (1LL << 15)   // 32^3: measured 62 against 79 us per step; 64^3 is a tie, 256 x 16 x 16 loses
#endif

template <int RC>
int launch_small(SmallArgs &a) {
  static int blocks_per_sm = -1;
  if (blocks_per_sm < 0) {
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, k_small_steps<RC>, 256, 0));
    if (blocks_per_sm < 1) return fail(MHD_ERR_CUDA, "k_small_steps does not fit on an SM");
  }
  const Geo &g = C.g;
  const int r = recon_radius(RC);
  long long work = 1;
  for (int x = 0; x < 3; x++) work *= (g.n[x] + 2 * r + 4);   // the largest phase: predictor fluxes
  long long blocks = (work + 255) / 256;
  const long long cap = (long long)blocks_per_sm * C.num_sms;   // co-resident blocks (grid barrier)
  if (blocks > cap) blocks = cap;
  void *args[] = {&a};
  CU(cudaLaunchCooperativeKernel((void *)k_small_steps<RC>, dim3((unsigned)blocks), dim3(256), args, 0, C.stream));
  LAUNCH_CHECK("k_small_steps");
  return MHD_OK;
}

// n steps of { dt = cfl / max rate (or dt_fixed); step } in one cooperative launch
int run_small(int n_steps, double cfl, double dt_fixed) {
  SmallArgs a;
  a.U = C.U; a.Uh = C.Uh; a.F = C.F; a.E = C.E; a.Er = C.Er; a.Bnext = C.Bnext; a.g = C.g; a.sc = C.sc;
  a.n_steps = n_steps; a.cfl = cfl; a.dt_fixed = dt_fixed;
  a.dbg = getenv("MHD_SMALL_DEBUG") ? (unsigned long long *)C.scratch : nullptr;
  int rc;
  switch (C.g.recon) {
    case 0: rc = launch_small<0>(a); break;
    case 1: rc = launch_small<1>(a); break;
    case 2: rc = launch_small<2>(a); break;
    case 3: rc = launch_small<3>(a); break;
    default: rc = launch_small<4>(a); break;
  }
  if (rc) return rc;
  if (a.dbg) {
    unsigned long long h[16];
    cudaMemcpyAsync(h, a.dbg, sizeof(h), cudaMemcpyDeviceToHost, C.stream);
    cudaStreamSynchronize(C.stream);
    fprintf(stderr, "k_small_steps last step, us per phase (ghosts, pred flux, ct, half update, face flux, ct, update):");
    for (int q = 1; q < 8; q++) fprintf(stderr, " %.1f", (h[q] - h[q - 1]) * 1e-3);
    fprintf(stderr, "\n");
  }
  if (n_steps & 1) {   // the B ping-pong inside the kernel ended on the other set of face arrays
    for (int x = 0; x < 3; x++) { double *t = C.Bnext.f[x]; C.Bnext.f[x] = C.U.f[F_BX + x]; C.U.f[F_BX + x] = t; }
    C.parity ^= 1;
  }
  C.rate_valid = true;
  return MHD_OK;
}

}  // namespace

extern "C" {

size_t mhd_workspace_bytes(int nx, int ny, int nz, int recon) {
  Geo g;
  if (!make_geo(g, nx, ny, nz, 1.5, recon)) return 0;
  return total_bytes(g);
}

int mhd_init(int nx, int ny, int nz, double gamma, int recon) {
  return init_common(nx, ny, nz, gamma, recon, nullptr, 0);
}

int mhd_init_workspace(int nx, int ny, int nz, double gamma, int recon, void *workspace,
                       size_t workspace_bytes) {
  if (!workspace) return fail(MHD_ERR_ARG, "mhd_init_workspace: null workspace");
  return init_common(nx, ny, nz, gamma, recon, workspace, workspace_bytes);
}

int mhd_set_boundary(int axis, int kind) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (axis < 0 || axis > 2 || (kind != MHD_BC_PERIODIC && kind != MHD_BC_OUTFLOW))
    return fail(MHD_ERR_ARG, "mhd_set_boundary: bad argument");
  C.g.bc[axis] = kind;
  drop_graph();
  return MHD_OK;
}

int mhd_set_domain(double lx, double ly, double lz) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  const double L[3] = {lx, ly, lz};
  for (int a = 0; a < 3; a++)
    if (!(L[a] > 0.0)) return fail(MHD_ERR_ARG, "mhd_set_domain: lengths must be positive");
  for (int a = 0; a < 3; a++) { C.g.d[a] = L[a] / C.g.n[a]; C.g.id[a] = C.g.n[a] / L[a]; }
  drop_graph();
  C.rate_valid = false;
  return MHD_OK;
}

int mhd_set_stream(void *cuda_stream) {
  if (C.stream != (cudaStream_t)cuda_stream) drop_graph();
  C.stream = (cudaStream_t)cuda_stream;
  return MHD_OK;
}

int mhd_set_state(const double *rho, const double *mx, const double *my, const double *mz,
                  const double *E, const double *bx, const double *by, const double *bz) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  const double *src[NFIELD] = {rho, mx, my, mz, E, bx, by, bz};
  int rc = set_state_from(src, true);
  if (rc) return rc;
  CU(cudaStreamSynchronize(C.stream));
  return MHD_OK;
}

int mhd_set_state_device(const double *rho, const double *mx, const double *my, const double *mz,
                         const double *E, const double *bx, const double *by, const double *bz) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  const double *src[NFIELD] = {rho, mx, my, mz, E, bx, by, bz};
  return set_state_from(src, false);
}

int mhd_compute_dt(double cfl, double *dt) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (!dt || !(cfl > 0.0)) return fail(MHD_ERR_ARG, "mhd_compute_dt: bad argument");
  int rc = ensure_rate();
  if (rc) return rc;
  Scalars h;
  CU(cudaMemcpyAsync(&h, C.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, C.stream));
  CU(cudaStreamSynchronize(C.stream));
  double m;
  memcpy(&m, &h.rate_bits, sizeof(double));
  *dt = cfl / m;
  if (h.bad) return fail(MHD_ERR_UNPHYSICAL, "non-physical state (rho <= 0, P <= 0 or non-finite)");
  return MHD_OK;
}

int mhd_step(double dt) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (!(dt > 0.0)) return fail(MHD_ERR_ARG, "mhd_step: dt must be positive");
  if (C.small_mode == 1 && C.coop && C.prof_n < 0) return run_small(1, 1.0, dt);
  k_set_dt<<<1, 1, 0, C.stream>>>(C.sc, dt);
  LAUNCH_CHECK("k_set_dt");
  return step_kernels();
}

int mhd_advance(int n_steps, double cfl, double *t_accum) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (n_steps < 0 || !(cfl > 0.0)) return fail(MHD_ERR_ARG, "mhd_advance: bad argument");
  Scalars h;
  double t0 = 0.0;
  if (t_accum) {
    CU(cudaMemcpyAsync(&h, C.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, C.stream));
    CU(cudaStreamSynchronize(C.stream));
    t0 = h.t_accum;
  }
  int s = 0;
  const long long ncell = (long long)C.g.n[0] * C.g.n[1] * C.g.n[2];
  if (C.coop && C.prof_n < 0 && n_steps > 0 && (C.small_mode == 1 || (C.small_mode == 0 && ncell <= MHD_SMALL_MAX_CELLS))) {
    int rc = ensure_rate();
    if (rc) return rc;
    rc = run_small(n_steps, cfl, 0.0);
    if (rc) return rc;
    s = n_steps;
  }
  if (C.stream != 0 && n_steps - s >= 4 && ncell <= (1LL << 21) && C.prof_n < 0) {  // launch-bound sizes only
    int rc = ensure_rate();
    if (rc) return rc;
    const int p = C.parity;
    if (!C.graph[p] || C.graph_cfl[p] != cfl) {
      rc = build_graph(cfl);
      if (rc) return rc;
    }
    for (; s + 2 <= n_steps; s += 2) {
      CU(cudaGraphLaunch(C.graph[p], C.stream));
      C.launches += C.graph_launches;
    }
  }
  for (; s < n_steps; s++) {
    int rc = ensure_rate();
    if (rc) return rc;
    k_finish_dt<<<1, 1, 0, C.stream>>>(C.sc, cfl);
    LAUNCH_CHECK("k_finish_dt");
    rc = step_kernels();
    if (rc) return rc;
  }
  if (t_accum) {
    CU(cudaMemcpyAsync(&h, C.sc, sizeof(Scalars), cudaMemcpyDeviceToHost, C.stream));
    CU(cudaStreamSynchronize(C.stream));
    *t_accum = h.t_accum - t0;
    if (h.bad) return fail(MHD_ERR_UNPHYSICAL, "non-physical state (rho <= 0, P <= 0 or non-finite)");
  }
  return MHD_OK;
}

int mhd_get_state(double *rho, double *mx, double *my, double *mz, double *E, double *bx,
                  double *by, double *bz) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  double *dst[NFIELD] = {rho, mx, my, mz, E, bx, by, bz};
  int rc = get_state_to(C.U, dst, true);
  if (rc) return rc;
  CU(cudaStreamSynchronize(C.stream));
  return MHD_OK;
}

int mhd_get_state_device(double *rho, double *mx, double *my, double *mz, double *E, double *bx,
                         double *by, double *bz) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  double *dst[NFIELD] = {rho, mx, my, mz, E, bx, by, bz};
  return get_state_to(C.U, dst, false);
}

int mhd_get_half_state(double *rho, double *mx, double *my, double *mz, double *E, double *bx,
                       double *by, double *bz) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  double *dst[NFIELD] = {rho, mx, my, mz, E, bx, by, bz};
  // the half state is held as (rho, v, P, face B): convert to the ABI's conserved variables in
  // arrays that are dead after the step and exposed by no call (edge fields, B^n's old set)
  const Geo &g = C.g;
  State8 tmp = C.Uh;
  tmp.f[0] = C.E.f[0]; tmp.f[1] = C.E.f[1]; tmp.f[2] = C.E.f[2]; tmp.f[3] = C.Bnext.f[0]; tmp.f[4] = C.Bnext.f[1];
  Box ab = make_box(0, g.n[0] - 1, 0, g.n[1] - 1, 0, g.n[2] - 1);
  long long plane = (long long)g.n[0] * g.n[1];
  k_half_to_cons<<<dim3(grid1(plane, 256).x, g.n[2]), 256, 0, C.stream>>>(C.Uh, tmp, g, ab);
  LAUNCH_CHECK("k_half_to_cons");
  int rc = get_state_to(tmp, dst, true);
  if (rc) return rc;
  CU(cudaStreamSynchronize(C.stream));
  return MHD_OK;
}

int mhd_get_flux(int axis, int comp, double *out) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (axis < 0 || axis > 2 || comp < 0 || comp > 6 || !out) return fail(MHD_ERR_ARG, "mhd_get_flux: bad argument");
  if (axis == 2 && comp >= 1 && comp <= 4)
    return fail(MHD_ERR_ARG, "mhd_get_flux: the z momentum / energy fluxes are consumed in the z sweep, not stored");
  const Geo &g = C.g;
  long long cnt = (long long)g.n[0] * g.n[1] * g.n[2];
  double *stage = C.scratch;
  k_pack<<<grid1(cnt, 256), 256, 0, C.stream>>>(stage, C.F.f[axis][comp], g, g.n[0], g.n[1], g.n[2]);
  LAUNCH_CHECK("k_pack");
  CU(cudaMemcpyAsync(out, stage, cnt * sizeof(double), cudaMemcpyDeviceToHost, C.stream));
  CU(cudaStreamSynchronize(C.stream));
  return MHD_OK;
}

int mhd_max_divb(double *out) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (!out) return fail(MHD_ERR_ARG, "mhd_max_divb: null pointer");
  const Geo &g = C.g;
  unsigned long long *bits = (unsigned long long *)C.E.f[0];  // edge fields are free between steps
  CU(cudaMemsetAsync(bits, 0, sizeof(unsigned long long), C.stream));
  long long plane = (long long)g.n[0] * g.n[1];
  dim3 grid(grid1(plane, 256).x, g.n[2]);
  k_divb<<<grid, 256, 0, C.stream>>>(C.U, g, bits);
  LAUNCH_CHECK("k_divb");
  unsigned long long h;
  CU(cudaMemcpyAsync(&h, bits, sizeof(h), cudaMemcpyDeviceToHost, C.stream));
  CU(cudaStreamSynchronize(C.stream));
  memcpy(out, &h, sizeof(double));
  return MHD_OK;
}

// n_steps steps with a CUDA event after every launch, all enqueued back to back (no synchronisation
// until the last one), then the duration of launch i of a step averaged over the steps.
// cfl > 0: every step takes its own dt from the CFL reduction, as mhd_advance does; else the given dt.
int profiled_steps(int n_steps, double dt, double cfl, int max_entries, double *ms, const char **names, int *n_entries) {
  const int cap = kMaxProf * n_steps;
  std::vector<cudaEvent_t> ev((size_t)cap + 1, nullptr);
  std::vector<const char *> nm((size_t)cap, nullptr);
  int rc = MHD_OK;
  for (auto &e : ev)
    if (!rc && cudaEventCreate(&e) != cudaSuccess) rc = fail(MHD_ERR_CUDA, "cudaEventCreate failed");
  auto enqueue = [&]() -> int {
    if (cfl > 0.0) {
      int r = ensure_rate();
      if (r) return r;
    } else {
      k_set_dt<<<1, 1, 0, C.stream>>>(C.sc, dt);
      LAUNCH_CHECK("k_set_dt");
    }
    C.prof_ev = ev.data(); C.prof_name = nm.data(); C.prof_cap = cap;
    C.prof_n = 0;
    cudaEventRecord(ev[0], C.stream);
    for (int s = 0; s < n_steps; s++) {
      if (cfl > 0.0) {
        k_finish_dt<<<1, 1, 0, C.stream>>>(C.sc, cfl);
        LAUNCH_CHECK("k_finish_dt");
      }
      int r = step_kernels();
      if (r) return r;
    }
    return MHD_OK;
  };
  if (!rc) rc = enqueue();
  const int n = C.prof_n;
  C.prof_n = -1; C.prof_cap = 0; C.prof_ev = nullptr; C.prof_name = nullptr;
  cudaError_t e = cudaStreamSynchronize(C.stream);
  if (!rc && e != cudaSuccess) rc = cuda_fail(e, "cudaStreamSynchronize");
  *n_entries = 0;
  if (!rc && n > 0 && n % n_steps == 0) {
    const int per = n / n_steps;
    for (int i = 0; i < per && i < max_entries; i++) {
      double sum = 0.0;
      for (int s = 0; s < n_steps; s++) {
        float t = 0.f;
        cudaEventElapsedTime(&t, ev[(size_t)s * per + i], ev[(size_t)s * per + i + 1]);
        sum += t;
      }
      ms[i] = sum / n_steps; names[i] = nm[i]; *n_entries = i + 1;
    }
  } else if (!rc) {
    rc = fail(MHD_ERR_CUDA, "profiled steps recorded an unexpected number of launches");
  }
  for (auto &x : ev)
    if (x) cudaEventDestroy(x);
  return rc;
}

int mhd_step_profile(double dt, int max_entries, double *ms, const char **names, int *n_entries) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (!(dt > 0.0) || !ms || !names || !n_entries || max_entries < 1)
    return fail(MHD_ERR_ARG, "mhd_step_profile: bad argument");
  return profiled_steps(1, dt, 0.0, max_entries, ms, names, n_entries);
}

int mhd_advance_profile(int n_steps, double cfl, int max_entries, double *ms, const char **names, int *n_entries) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (n_steps < 1 || n_steps > 4096 || !(cfl > 0.0) || !ms || !names || !n_entries || max_entries < 1)
    return fail(MHD_ERR_ARG, "mhd_advance_profile: bad argument");
  return profiled_steps(n_steps, 0.0, cfl, max_entries, ms, names, n_entries);
}

int mhd_debug_guard_errors(long long *n_bad) {
  if (!C.inited) return fail(MHD_ERR_NOT_INIT, "not initialised");
  if (!n_bad) return fail(MHD_ERR_ARG, "mhd_debug_guard_errors: null pointer");
  *n_bad = -1;
  if (!C.guard) return MHD_OK;   // not a guarded context
  unsigned long long *cnt = (unsigned long long *)&C.sc[1];   // (the scalar block is 256 bytes)
  CU(cudaMemsetAsync(cnt, 0, sizeof(*cnt), C.stream));
  const size_t slot = (array_bytes(C.g) + 2 * C.guard) / 8;
  k_count_guard_damage<<<512, 256, 0, C.stream>>>((const unsigned long long *)((char *)C.base + 256), slot, C.guard / 8,
                                                  kNumArrays, kGuardPattern, cnt);
  LAUNCH_CHECK("k_count_guard_damage");
  unsigned long long h = 0;
  CU(cudaMemcpyAsync(&h, cnt, sizeof(h), cudaMemcpyDeviceToHost, C.stream));
  CU(cudaStreamSynchronize(C.stream));
  *n_bad = (long long)h;
  return MHD_OK;
}

long long mhd_launch_count(void) { return C.launches; }

int mhd_synchronize(void) {
  CU(cudaStreamSynchronize(C.stream));
  return MHD_OK;
}

int mhd_finalize(void) {
  if (C.inited) {
    cudaStreamSynchronize(C.stream);
    drop_graph();
    if (C.owns_memory && C.base) cudaFree(C.base);
  }
  cudaStream_t s = C.stream;
  C = Context();
  C.stream = s;
  return MHD_OK;
}

const char *mhd_last_error(void) { return g_err; }

}  // extern "C"
