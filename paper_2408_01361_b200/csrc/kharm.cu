// kharm.cu -- C ABI (include/kharm.h) and host orchestration of the HARM step on one B200.
// All arithmetic of the path runs in the kernels of kh_kernels.cuh / kh_geometry.cuh; the host
// only validates arguments, owns device buffers and enqueues launches on the grid's stream.
#include "../../include/kharm.h"

#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <new>

#include <nvtx3/nvToolsExt.h>      // header-only; ranges are no-ops unless a tool is attached

#include "kh_geometry.cuh"
#include "kh_kernels.cuh"

using namespace kh;

static thread_local char g_cuda_err[256] = "";

#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      snprintf(g_cuda_err, sizeof(g_cuda_err), "%s at %s:%d", cudaGetErrorString(e_), __FILE__, __LINE__); \
      return (e_ == cudaErrorMemoryAllocation) ? KH_ENOMEM : KH_ECUDA;                             \
    }                                                                                              \
  } while (0)

enum { KH_GP_MAX = 64 };

struct kh_grid {
  kh_params p;
  GV gv;
  cudaStream_t stream;
  bool own_stream;
  bool flat;
  // device buffers
  double* geom[4];
  double* conn;
  double* dg;
  double* floorp;
  double* P[3];          // P^n, P*, P^{n+1} (rotating)
  double* F[3];          // face fluxes per direction, [8][ntot]
  double* ctop[3];
  double* emf[3];
  unsigned char *pflag, *fflag;
  double* ecent[4];      // upwinded EMFs: zone-centred reference values + conserved density (allocated on demand)
  bool faces_set;        // face-centred CT: kh_set_face_B has been called (the face field is the magnetic state from then on)
  bool has_fixed;        // some boundary is KH_BC_FIXED ...
  bool fixed_ghosts_set; // ... and a with_ghosts = 1 load has supplied the ghost layers
  bool have_dt_next;     // a completed step has left a dt_next on the device (kh_step(dt <= 0) is legal)
  int device;            // the CUDA device the grid lives on
  bool has_block;        // some side is KH_BC_BLOCK: stepped by kh_step_blocks only
  kh_grid* nb[3][2];     // neighbouring block across [dir - 1][side] (kh_link_blocks)
  double* halo_buf[3][2];// message buffer of the 3 layers next to that side: [9][3][t2][t1] doubles (8 primitives + flag)
  double* Bf[3][3];      // face-centred CT: Phi^d per rotation state [state][d], [ntot] each (allocated on demand)
  unsigned char* mask;   // FOFC: troubled zones of the speculative update (with ghost images)
  unsigned* faillist;    // zones (device-layout index) whose inversion failed in the current sub-step
  double* fix;           // [5][ntot] scratch of the fix-up (pre-fix-up snapshot semantics)
  double* stage;         // lazily allocated [8][ntot] staging buffer for host transfers / debug copies
  StepScalars* sc;       // device
  StepScalars* sc_host;  // pinned
  int cur;               // index of P^n in P[]
  long long launches;
  // CUDA graphs of a full step, one per rotation state of the P buffers
  bool use_graph;
  cudaGraphExec_t gexec[3];
  long long graph_launches;   // kernel launches inside one captured step
  // per-kernel timing (kh_set_profile): event pairs around every launch, summed per kind on read-out
  bool profile;
  cudaEvent_t* pev;           // 2 * KH_PROF_POOL events
  int* pkind;
  int npev;
  int sm_count, flux_blocks_per_sm;
  // the three flux directions of a sub-step are independent: x2 and x3 run on two side streams (fork / join by events,
  // captured into the step's graph), so that the last partial wave of one kernel is filled by the blocks of the next
  cudaStream_t side[2];
  cudaEvent_t ev_fork, ev_join[2];
  bool flux_concurrent;
  bool update_tma;            // update_tma_kernel (needs an even padded row length) instead of update_kernel
  // tensor maps of the update kernel's tile copies (cuTensorMapEncodeTiled, once per grid): one per array and box shape
  CUtensorMap mapF[3], mapE[3], mapP[3], mapBf[3][3], mapT[3];     // mapT: centre geometry, source and floor tables
  int march_J;                // 0 = chosen by march_chunk()
  double prof_ms[KH_K_COUNT];
  long long prof_n[KH_K_COUNT];
  // profiling INSIDE the step's graph: event-record nodes (cudaEventRecordExternal) around every launch group of a second,
  // instrumented graph per rotation state, read out after each replay -- the timed kernels then run exactly as in the product
  // path (the concurrent flux directions overlap as they do there; direct launches bracketed by events do not reproduce that)
  cudaGraphExec_t gexec_prof[3];
  cudaEvent_t gpev[3][KH_GP_MAX][2];
  int gpkind[3][KH_GP_MAX];
  int gpn[3];
  int gp_capture;             // rotation state + 1 while an instrumented graph is being captured, else 0
};

enum { KH_PROF_POOL = 2048 };

static void prof_flush(kh_grid* g) {
  if (!g->npev) return;
  cudaEventSynchronize(g->pev[2 * (g->npev - 1) + 1]);
  for (int r = 0; r < g->npev; r++) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, g->pev[2 * r], g->pev[2 * r + 1]) == cudaSuccess) {
      g->prof_ms[g->pkind[r]] += ms;
      g->prof_n[g->pkind[r]]++;
    }
  }
  g->npev = 0;
}
struct NvtxRange { explicit NvtxRange(const char* n) { nvtxRangePushA(n); } ~NvtxRange() { nvtxRangePop(); } };
static const char* const kKindName[KH_K_COUNT] = {"kh:flux", "kh:flux2", "kh:flux3", "kh:emf", "kh:update", "kh:fill", "kh:fixup", "kh:fofc"};
// bracket one launch group: prof_begin(kind); kernel<<<...>>>(...); prof_end();  Always an NVTX range (host side: it marks the
// enqueue, or the capture, of the group); with kh_set_profile also a pair of CUDA events.
static inline void prof_begin(kh_grid* g, int kind) {
  nvtxRangePushA(kKindName[kind]);
  if (!g->profile) return;
  if (g->gp_capture) {
    const int c = g->gp_capture - 1, r = g->gpn[c];
    if (r >= KH_GP_MAX) return;
    if (!g->gpev[c][r][0]) { cudaEventCreate(&g->gpev[c][r][0]); cudaEventCreate(&g->gpev[c][r][1]); }
    g->gpkind[c][r] = kind;
    cudaEventRecordWithFlags(g->gpev[c][r][0], g->stream, cudaEventRecordExternal);
    return;
  }
  if (g->npev == KH_PROF_POOL) prof_flush(g);
  g->pkind[g->npev] = kind;
  cudaEventRecord(g->pev[2 * g->npev], g->stream);
}
static inline void prof_end(kh_grid* g) {
  nvtxRangePop();
  if (!g->profile) return;
  if (g->gp_capture) {
    const int c = g->gp_capture - 1, r = g->gpn[c];
    if (r >= KH_GP_MAX) return;
    cudaEventRecordWithFlags(g->gpev[c][r][1], g->stream, cudaEventRecordExternal);
    g->gpn[c]++;
    return;
  }
  cudaEventRecord(g->pev[2 * g->npev + 1], g->stream);
  g->npev++;
}

static inline dim3 zone_grid(int nx, int ny, int nz) { return dim3((nx + 127) / 128, ny, nz); }

static int fill_ghosts(kh_grid* g, double* P, unsigned char* flag) {
  const GV& v = g->gv;
  const long shell = (long)v.nt1 * v.nt2 * (2 * KH_NGH) + (long)v.nt1 * (2 * KH_NGH) * v.n3 + (long)(2 * KH_NGH) * v.n2 * v.n3;
  prof_begin(g, KH_K_FILL);
  fill_kernel<<<(unsigned)((shell + 127) / 128), 128, 0, g->stream>>>(v, P, flag);
  prof_end(g);
  g->launches += 1;
  CK(cudaGetLastError());
  return KH_OK;
}

// The marching kernels stage their stencil rows through a shared-memory ring: ask for the large carve-out so that
// several blocks stay resident (B200: up to 227 KB of shared memory per SM).
template <int DIR, int RECON, bool FLAT>
static void setup_march_one() {
  cudaFuncSetAttribute(flux_march_kernel<DIR, RECON, FLAT>, cudaFuncAttributeMaxDynamicSharedMemorySize, MarchRing<RECON>::BYTES);
  cudaFuncSetAttribute(flux_march_kernel<DIR, RECON, FLAT>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}
static void setup_march_kernels() {
  setup_march_one<2, 0, true>(); setup_march_one<2, 1, true>(); setup_march_one<2, 0, false>(); setup_march_one<2, 1, false>();
  setup_march_one<3, 0, true>(); setup_march_one<3, 1, true>(); setup_march_one<3, 0, false>(); setup_march_one<3, 1, false>();
}

// A tensor map over one zone array as ALLOCATED (the array proper starts one double later: TileMaps): rank 3 (nt1, nt2, nt3) or,
// with nvar > 1, rank 4 (nt1, nt2, nt3, nvar); box = the tile's box.  false if the driver entry point or the encoding fails.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) fn = (EncodeTiledFn)p;
    cudaGetLastError();
  }
  return fn;
}
static bool make_tile_map(CUtensorMap* map, const double* array, const GV& v, int nvar, int b0, int b1, int b2) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  const cuuint32_t rank = nvar > 1 ? 4 : 3;
  cuuint64_t dims[4] = {(cuuint64_t)v.nt1, (cuuint64_t)v.nt2, (cuuint64_t)v.nt3, (cuuint64_t)nvar};
  cuuint64_t strides[3] = {(cuuint64_t)v.nt1 * 8, (cuuint64_t)v.s3 * 8, (cuuint64_t)v.ntot * 8};      // bytes, dimensions 1 .. rank - 1
  cuuint32_t box[4] = {(cuuint32_t)b0, (cuuint32_t)b1, (cuuint32_t)b2, (cuuint32_t)nvar};
  cuuint32_t es[4] = {1, 1, 1, 1};
  return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, rank, (void*)(array - 1), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// a table of `comps` components over the padded (x1, x2) plane: box = 32 zones of one row, all components.  Like the zone arrays
// the table starts one double past its allocation, which is what the map describes: every box then starts on a 16 B boundary
// (a box starting 8 B off one raises an illegal-instruction fault on sm_100a)
static bool make_table_map(CUtensorMap* map, const double* table, const GV& v, int comps) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {(cuuint64_t)v.nt1, (cuuint64_t)v.nt2, (cuuint64_t)comps};
  cuuint64_t strides[2] = {(cuuint64_t)v.nt1 * 8, (cuuint64_t)v.n2d * 8};
  cuuint32_t box[3] = {32, 1, (cuuint32_t)comps};
  cuuint32_t es[3] = {1, 1, 1};
  return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)(table - 1), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
static bool make_tile_maps(kh_grid* g) {
  const GV& v = g->gv;
  if (!g->flat && !(make_table_map(&g->mapT[0], g->geom[0], v, KH_NGEO) && make_table_map(&g->mapT[1], g->dg, v, KH_NDG) &&
                    make_table_map(&g->mapT[2], g->floorp, v, 2)))
    return false;
  bool ok = make_tile_map(&g->mapF[0], g->F[0], v, 5, 34, 1, 1) && make_tile_map(&g->mapF[1], g->F[1], v, 5, 32, 2, 1) &&
            make_tile_map(&g->mapF[2], g->F[2], v, 5, 32, 1, 2);
  // e3 at (i, i+1) x (j, j+1); e2 at (i, i+1) x (k, k+1); e1 at (j, j+1) x (k, k+1)
  ok = ok && make_tile_map(&g->mapE[2], g->emf[2], v, 1, 34, 2, 1) && make_tile_map(&g->mapE[1], g->emf[1], v, 1, 34, 1, 2) &&
       make_tile_map(&g->mapE[0], g->emf[0], v, 1, 32, 2, 2);
  for (int b = 0; b < 3 && ok; b++) ok = make_tile_map(&g->mapP[b], g->P[b], v, KH_NP, 32, 1, 1);
  if (g->p.transport == KH_B_FACE_CT)
    for (int b = 0; b < 3 && ok; b++)
      ok = make_tile_map(&g->mapBf[b][0], g->Bf[b][0], v, 1, 34, 1, 1) && make_tile_map(&g->mapBf[b][1], g->Bf[b][1], v, 1, 32, 2, 1) &&
           make_tile_map(&g->mapBf[b][2], g->Bf[b][2], v, 1, 32, 1, 2);
  return ok;
}

template <bool FL, bool CO, int MODE>
static constexpr size_t tile_smem_bytes() {     // one tile and one mbarrier per warp, two geometry buffers with their barriers and counters, alignment to 128 B
  return KH_UPD_WARPS * ((size_t)TileLayout<FL, CO, MODE>::BYTES + 8) + (FL ? 0 : 2 * (size_t)KH_GEO_ROWS * 32 * 8) + 32 + 128;
}
template <bool FL, bool CO, int MODE>
static cudaError_t setup_update_tma_one() {
  cudaError_t e = cudaFuncSetAttribute(update_tma_kernel<FL, CO, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem_bytes<FL, CO, MODE>());
  if (e == cudaSuccess) e = cudaFuncSetAttribute(update_tma_kernel<FL, CO, MODE>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  return e;
}
template <int MODE>
static cudaError_t setup_update_tma_mode(bool flat) {
  cudaError_t e = flat ? setup_update_tma_one<true, false, MODE>() : setup_update_tma_one<false, false, MODE>();
  if (e == cudaSuccess) e = flat ? setup_update_tma_one<true, true, MODE>() : setup_update_tma_one<false, true, MODE>();
  return e;
}
static cudaError_t setup_update_tma(bool flat, int mode) {
  switch (mode) {
    case 0: return setup_update_tma_mode<0>(flat); case 1: return setup_update_tma_mode<1>(flat);
    case 2: return setup_update_tma_mode<2>(flat); case 3: return setup_update_tma_mode<3>(flat);
    case 4: return setup_update_tma_mode<4>(flat); case 5: return setup_update_tma_mode<5>(flat);
    case 8: return setup_update_tma_mode<8>(flat); case 9: return setup_update_tma_mode<9>(flat);
    case 10: return setup_update_tma_mode<10>(flat); case 11: return setup_update_tma_mode<11>(flat);
    case 12: return setup_update_tma_mode<12>(flat); default: return setup_update_tma_mode<13>(flat);
  }
}

// Chunk length of the marching kernels: long enough that the one extra reconstruction per chunk is
// small, short enough that the grid fills the SMs in an almost whole number of waves.
static int march_chunk(const kh_grid* g, long columns, int faces) {
  const double resident = (double)g->sm_count * g->flux_blocks_per_sm * 128.0;
  int best = 16;
  double best_eff = 0.0;
  for (int J = 6; J <= 32; J++) {
    int chunks = (faces + J - 1) / J;
    double waves = (double)columns * chunks / resident;
    double eff = waves / ceil(waves) * ((double)faces / (double)(faces + chunks));
    if (eff > best_eff + 1e-9) { best_eff = eff; best = J; }
  }
  return best;
}

template <int DIR>
static void launch_flux(kh_grid* g, const double* Ps, cudaStream_t stream, bool prof) {
  const GV& v = g->gv;
  double* F = g->F[DIR - 1];
  double* ct = g->ctop[DIR - 1];
  const bool mc = g->p.recon == KH_RECON_MC;
  if (prof) prof_begin(g, KH_K_FLUX1 + DIR - 1);
  if (DIR == 1) {
    const long zones = (long)(v.n1 + 2) * (v.thi2 - v.tlo2) * (v.thi3 - v.tlo3);
    const long warps = (zones + 30) / 31;
    const unsigned blocks = (unsigned)((warps + 3) / 4);
    if (g->flat) {
      if (mc) flux_x1_kernel<0, true><<<blocks, 128, 0, stream>>>(v, Ps, F, ct);
      else flux_x1_kernel<1, true><<<blocks, 128, 0, stream>>>(v, Ps, F, ct);
    } else {
      if (mc) flux_x1_kernel<0, false><<<blocks, 128, 0, stream>>>(v, Ps, F, ct);
      else flux_x1_kernel<1, false><<<blocks, 128, 0, stream>>>(v, Ps, F, ct);
    }
  } else {
    const int N = (DIR == 2) ? v.n2 : v.n3;
    const long cols = (long)(v.n1 + 2) * (DIR == 2 ? v.thi3 - v.tlo3 : v.thi2 - v.tlo2);
    // concurrent directions: whole columns (no redundant reconstruction at chunk starts; the x1 kernel's many small blocks fill
    // the SMs the few long-running marching blocks leave free); alone: chunks that fill the SMs in whole waves
    int J;
    if (g->march_J > 0) J = g->march_J;
    else if (g->flux_concurrent) {
      // a marching thread is a serial chain of J faces (~5300 cycles each when the SM is full) that must not outlast the
      // whole group (3 Z zone-faces at ~2000 cycles per warp-face on 4 x SMs sub-partitions): J <= ~6e-5 Z
      const double Z = (double)(v.n1 + 2) * (v.n2 + 2) * (v.n3 + 2);
      const int jmax = (int)(Z * (3.0 * 2000.0 / (32.0 * 5300.0)) / (4.0 * g->sm_count));
      const int chunks = (N + 1 + (jmax > 8 ? jmax : 8) - 1) / (jmax > 8 ? jmax : 8);
      J = (N + 1 + chunks - 1) / chunks;
    } else J = march_chunk(g, cols, N + 1);
    dim3 grid((unsigned)((cols + 127) / 128), (unsigned)((N + 1 + J - 1) / J));
    constexpr int D = (DIR == 1) ? 2 : DIR;   // (keeps the DIR == 1 instantiation of this branch well-formed)
    const size_t sm0 = MarchRing<0>::BYTES, sm1 = MarchRing<1>::BYTES;
    if (g->flat) {
      if (mc) flux_march_kernel<D, 0, true><<<grid, 128, sm0, stream>>>(v, Ps, F, ct, J);
      else flux_march_kernel<D, 1, true><<<grid, 128, sm1, stream>>>(v, Ps, F, ct, J);
    } else {
      if (mc) flux_march_kernel<D, 0, false><<<grid, 128, sm0, stream>>>(v, Ps, F, ct, J);
      else flux_march_kernel<D, 1, false><<<grid, 128, sm1, stream>>>(v, Ps, F, ct, J);
    }
  }
  if (prof) prof_end(g);
  g->launches++;
}

// Fix-up of the zones on the failure list (+ floors, + their ghost images).
static int do_fixup(kh_grid* g, double* Pf, bool gathered = false) {
  const GV& v = g->gv;
  prof_begin(g, KH_K_FIXUP);
  if (!gathered) fixup_gather_kernel<<<64, 128, 0, g->stream>>>(v, Pf, g->pflag, g->faillist, g->fix, g->sc);
  if (g->flat) fixup_apply_kernel<true><<<64, 128, 0, g->stream>>>(v, Pf, g->faillist, g->fflag, g->fix, g->sc);
  else fixup_apply_kernel<false><<<64, 128, 0, g->stream>>>(v, Pf, g->faillist, g->fflag, g->fix, g->sc);
  prof_end(g);
  g->launches += gathered ? 1 : 2;
  CK(cudaGetLastError());
  return KH_OK;
}

// Ghost fill of the sub-step's result together with the fix-up's gather (fill_gather_kernel)
static int fill_ghosts_and_gather(kh_grid* g, double* Pf) {
  const GV& v = g->gv;
  const long shell = (long)v.nt1 * v.nt2 * (2 * KH_NGH) + (long)v.nt1 * (2 * KH_NGH) * v.n3 + (long)(2 * KH_NGH) * v.n2 * v.n3;
  prof_begin(g, KH_K_FILL);
  fill_gather_kernel<<<(unsigned)((shell + 127) / 128) + 64u, 128, 0, g->stream>>>(v, Pf, g->pflag, g->faillist, g->fix, g->sc, 64u);
  prof_end(g);
  g->launches += 1;
  CK(cudaGetLastError());
  return KH_OK;
}

// One sub-step (S22): fluxes from Ps, update of U(Pi), inversion with guess Pi, floors, fill, fix-up, fill.
static int substep(kh_grid* g, const double* Pi, const double* Ps, double* Pf, double dt_factor, bool corrector,
                   double* const* Bfi = nullptr, double* const* Bff = nullptr, bool with_fixup = true) {
  const GV& v = g->gv;
  // One thread's worth of work, but also the SINGLE predecessor of the three flux kernels in the step's graph.  Measured (r02):
  // with the reset folded into another kernel the predictor's flux kernels become root nodes of the graph, the executor
  // launches x1 first, its short blocks take every slot before the marching blocks are placed, and the step costs 9 % more
  // (1.66 -> 1.81 ms); a higher priority of the side streams does not change that.
  reset_counters_kernel<<<1, 1, 0, g->stream>>>(g->sc, 0);
  g->launches++;
  if (g->flux_concurrent) {
    // fork: x2 and x3 on the side streams, x1 (many short blocks, launched last: it fills what the marching blocks leave free)
    // on the grid's stream; join.  Profiling brackets the group as one entry (kind flux1), since the three overlap.
    prof_begin(g, KH_K_FLUX1);
    CK(cudaEventRecord(g->ev_fork, g->stream));
    for (int s = 0; s < 2; s++) CK(cudaStreamWaitEvent(g->side[s], g->ev_fork, 0));
    launch_flux<2>(g, Ps, g->side[0], false);
    launch_flux<3>(g, Ps, g->side[1], false);
    launch_flux<1>(g, Ps, g->stream, false);      // measured: x1 first costs 13 % of the step (its blocks then fill every slot)
    for (int s = 0; s < 2; s++) {
      CK(cudaEventRecord(g->ev_join[s], g->side[s]));
      CK(cudaStreamWaitEvent(g->stream, g->ev_join[s], 0));
    }
    prof_end(g);
  } else {
    launch_flux<1>(g, Ps, g->stream, true);
    launch_flux<2>(g, Ps, g->stream, true);
    launch_flux<3>(g, Ps, g->stream, true);
  }
  const int passes = g->p.fofc ? 2 : 1;       // FOFC: a speculative update first, then the re-flux, then the real one
  for (int pass = 0; pass < passes; pass++) {
    prof_begin(g, KH_K_EMF);
    if (g->p.emf != KH_EMF_ARITHMETIC) {
      if (g->flat) ecent_kernel<true><<<zone_grid(v.n1 + 2, v.n2 + 2, v.n3 + 2), 128, 0, g->stream>>>(v, Ps, g->ecent[0], g->ecent[1], g->ecent[2], g->ecent[3]);
      else ecent_kernel<false><<<zone_grid(v.n1 + 2, v.n2 + 2, v.n3 + 2), 128, 0, g->stream>>>(v, Ps, g->ecent[0], g->ecent[1], g->ecent[2], g->ecent[3]);
      if (g->p.emf == KH_EMF_UPWIND)
        emf_upwind_kernel<false><<<zone_grid(v.n1 + 1, v.n2 + 1, v.n3 + 1), 128, 0, g->stream>>>(v, g->F[0], g->F[1], g->F[2], g->ecent[0], g->ecent[1],
                                                                                                 g->ecent[2], g->ecent[3], g->emf[0], g->emf[1], g->emf[2]);
      else
        emf_upwind_kernel<true><<<zone_grid(v.n1 + 1, v.n2 + 1, v.n3 + 1), 128, 0, g->stream>>>(v, g->F[0], g->F[1], g->F[2], g->ecent[0], g->ecent[1],
                                                                                                g->ecent[2], g->ecent[3], g->emf[0], g->emf[1], g->emf[2]);
      g->launches++;
    } else {
      emf_kernel<<<dim3((unsigned)(((long)(v.n1 + 1) * (v.n2 + 1) + 127) / 128), (unsigned)(v.n3 + 1)), 128, 0, g->stream>>>(v, g->F[0], g->F[1], g->F[2], g->emf[0], g->emf[1], g->emf[2]);
    }
    prof_end(g);
    g->launches++;
    const double *fb1 = nullptr, *fb2 = nullptr, *fb3 = nullptr;
    if (Bfi && pass + 1 == passes) {
      // face-centred CT: advance the face field by the EMF circulation; the update then takes the zone's field from it
      prof_begin(g, KH_K_EMF);
      face_ct_kernel<<<zone_grid(v.n1 + 1, v.n2 + 1, v.n3 + 1), 128, 0, g->stream>>>(v, Bfi[0], Bfi[1], Bfi[2], Bff[0], Bff[1], Bff[2], g->emf[0],
                                                                                       g->emf[1], g->emf[2], g->sc, dt_factor);
      prof_end(g);
      g->launches++;
      CK(cudaGetLastError());
      fb1 = Bff[0]; fb2 = Bff[1]; fb3 = Bff[2];
    }
    const unsigned grid = (unsigned)(((long)v.n1 * v.n2 * v.n3 + 127) / 128);
    // persistent: one block of 16 warps per SM, never more blocks than there are work units (update_tma_kernel)
    const long tunits = (long)((v.n1 + 31) / 32) * v.n2 * ((v.n3 + 16 * KH_UPD_TPW - 1) / (16 * KH_UPD_TPW));
    const unsigned tgrid = (unsigned)(tunits < (long)g->sm_count ? tunits : (long)g->sm_count);
#define UPD_ARGS v, Pi, Ps, Pf, g->F[0], g->F[1], g->F[2], g->emf[0], g->emf[1], g->emf[2], g->ctop[0], g->ctop[1], g->ctop[2], g->pflag, \
                 g->fflag, g->faillist, g->sc, dt_factor, fb1, fb2, fb3
    TileMaps M;
    if (g->update_tma) {
      auto pbuf = [&](const double* q) { for (int b = 0; b < 3; b++) if (g->P[b] == q) return b; return 0; };
      M.f1 = g->mapF[0]; M.f2 = g->mapF[1]; M.f3 = g->mapF[2];
      M.geo = g->mapT[0]; M.dgt = g->mapT[1]; M.flo = g->mapT[2];
      M.pi = g->mapP[pbuf(Pi)]; M.ps = g->mapP[pbuf(Ps)];
      if (fb1) {
        int st = 0;
        for (int b = 0; b < 3; b++) if (g->Bf[b][0] == fb1) st = b;
        M.a = g->mapBf[st][0]; M.b = g->mapBf[st][1]; M.c = g->mapBf[st][2];
      } else {
        M.a = g->mapE[2]; M.b = g->mapE[1]; M.c = g->mapE[0];
      }
    }
#define UPD(FL, CO, IN)                                                                                       \
  do {                                                                                                        \
    if (g->update_tma)                                                                                        \
      update_tma_kernel<FL, CO, IN><<<tgrid, 32 * KH_UPD_WARPS, tile_smem_bytes<FL, CO, IN>(), g->stream>>>(v, M, Pi, Pf, g->ctop[0], g->ctop[1], g->ctop[2], \
                                                                                               g->pflag, g->fflag, g->faillist, g->sc, dt_factor); \
    else update_kernel<FL, CO, IN><<<grid, 128, 0, g->stream>>>(UPD_ARGS);                                   \
  } while (0)
    prof_begin(g, KH_K_UPDATE);
#define UPD2(FL, CO)                                                                 \
    switch (g->p.inverter + 2 * g->p.floor_frame + (fb1 ? 8 : 0)) {                  \
      case 0: UPD(FL, CO, 0); break; case 1: UPD(FL, CO, 1); break;                  \
      case 2: UPD(FL, CO, 2); break; case 3: UPD(FL, CO, 3); break;                  \
      case 4: UPD(FL, CO, 4); break; case 5: UPD(FL, CO, 5); break;                  \
      case 8: UPD(FL, CO, 8); break; case 9: UPD(FL, CO, 9); break;                  \
      case 10: UPD(FL, CO, 10); break; case 11: UPD(FL, CO, 11); break;              \
      case 12: UPD(FL, CO, 12); break; default: UPD(FL, CO, 13); break;              \
    }
    if (g->flat) { if (corrector) { UPD2(true, true) } else { UPD2(true, false) } }
    else { if (corrector) { UPD2(false, true) } else { UPD2(false, false) } }
#undef UPD2
    prof_end(g);
#undef UPD
#undef UPD_ARGS
    g->launches++;
    CK(cudaGetLastError());
    if (pass + 1 < passes) {
      // troubled zones of the speculative update -> mask (+ ghost images) -> donor-cell LLF on their faces
      prof_begin(g, KH_K_FOFC);
      CK(cudaMemsetAsync(g->mask, 0, v.ntot, g->stream));
      fofc_mask_kernel<<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, g->pflag, g->fflag, g->mask);
      prof_end(g);
      int rc = fill_ghosts(g, nullptr, g->mask);
      if (rc) return rc;
      prof_begin(g, KH_K_FOFC);
      if (g->flat) fofc_reflux_kernel<true><<<zone_grid(v.n1 + 2, v.n2 + 2, v.n3 + 2), 128, 0, g->stream>>>(v, Ps, g->mask, g->F[0], g->F[1], g->F[2], g->ctop[0], g->ctop[1], g->ctop[2]);
      else fofc_reflux_kernel<false><<<zone_grid(v.n1 + 2, v.n2 + 2, v.n3 + 2), 128, 0, g->stream>>>(v, Ps, g->mask, g->F[0], g->F[1], g->F[2], g->ctop[0], g->ctop[1], g->ctop[2]);
      reset_counters_kernel<<<1, 1, 0, g->stream>>>(g->sc, 1);
      prof_end(g);
      g->launches += 3;
      CK(cudaGetLastError());
    }
  }
  if (!with_fixup) return fill_ghosts(g, Pf, g->pflag);          // linked blocks: halo exchange, fix-up, halo exchange follow (kh_step_blocks)
  int rc = fill_ghosts_and_gather(g, Pf);
  if (rc) return rc;
  return do_fixup(g, Pf, true);      // also refreshes the ghost images of the fixed zones (the second fill of S22)
}

static int enqueue_step(kh_grid* g, int cur) {
  double *Pn = g->P[cur], *Pstar = g->P[(cur + 1) % 3], *Pnew = g->P[(cur + 2) % 3];
  const bool face = g->p.transport == KH_B_FACE_CT;
  int rc = substep(g, Pn, Pn, Pstar, 0.5, false, face ? g->Bf[cur] : nullptr, face ? g->Bf[(cur + 1) % 3] : nullptr);
  if (rc) return rc;
  rc = substep(g, Pn, Pstar, Pnew, 1.0, true, face ? g->Bf[cur] : nullptr, face ? g->Bf[(cur + 2) % 3] : nullptr);
  if (rc) return rc;
  finalize_dt_kernel<<<1, 1, 0, g->stream>>>(g->sc, g->p.cfl, g->p.dt_growth_max);
  g->launches++;
  CK(cudaGetLastError());
  return KH_OK;
}

static int ensure_stage(kh_grid* g) {
  if (g->stage) return KH_OK;
  size_t a = sizeof(double) * KH_NP * g->gv.ntot, b = sizeof(double) * 64 * g->gv.n2d;
  CK(cudaMalloc((void**)&g->stage, a > b ? a : b));
  return KH_OK;
}

// Every entry point runs on the grid's device, whatever device the calling thread had current.
static int enter(kh_grid* g) {
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev != g->device) CK(cudaSetDevice(g->device));
  return KH_OK;
}
#define ENTER(g) do { int rc_ = enter(g); if (rc_) return rc_; } while (0)

static void destroy_graphs(kh_grid* g) {
  for (int c = 0; c < 3; c++) {
    if (g->gexec[c]) { cudaGraphExecDestroy(g->gexec[c]); g->gexec[c] = nullptr; }
    if (g->gexec_prof[c]) { cudaGraphExecDestroy(g->gexec_prof[c]); g->gexec_prof[c] = nullptr; }
    g->gpn[c] = 0;
  }
}

// The zone arrays start ONE DOUBLE past the (256 B aligned) allocation: with 3 ghost zones per side, interior zone i = 0 of every
// row then sits on a 16 B boundary whenever the padded row length is even, which is what the TMA bulk copies of
// update_tma_kernel need (source address and size multiples of 16 B).
static void free_shifted(double* p) { if (p) cudaFree(p - 1); }

extern "C" {

const char* kh_strerror(int code) {
  switch (code) {
    case KH_OK: return "ok";
    case KH_EINVAL: return "invalid argument";
    case KH_ENOMEM: return "out of memory";
    case KH_ECUDA: return "CUDA error (see kh_last_cuda_error)";
    case KH_ENAN: return "non-finite value";
    case KH_ESIZE: return "problem larger than the static scratch of the allocation-free entry point (KH_NOALLOC_MAX_CORNERS)";
    default: return "unknown error";
  }
}
const char* kh_last_cuda_error(void) { return g_cuda_err; }

int kh_grid_destroy(kh_grid* g) {
  if (!g) return KH_OK;
  destroy_graphs(g);
  free_shifted(g->geom[0]);
  for (int l = 1; l < 4; l++) cudaFree(g->geom[l]);
  cudaFree(g->conn); free_shifted(g->dg); free_shifted(g->floorp);
  for (int b = 0; b < 3; b++) { free_shifted(g->P[b]); free_shifted(g->F[b]); free_shifted(g->ctop[b]); free_shifted(g->emf[b]); }
  cudaFree(g->pflag); cudaFree(g->fflag); cudaFree(g->mask);
  for (int b = 0; b < 3; b++) for (int d = 0; d < 3; d++) free_shifted(g->Bf[b][d]);
  for (int d = 0; d < 3; d++) for (int sd = 0; sd < 2; sd++) {
    cudaFree(g->halo_buf[d][sd]);
    if (g->nb[d][sd] && g->nb[d][sd]->nb[d][1 - sd] == g) g->nb[d][sd]->nb[d][1 - sd] = nullptr;    // unlink the neighbour
  }
  for (int d = 0; d < 4; d++) cudaFree(g->ecent[d]); cudaFree(g->faillist); cudaFree(g->sc); cudaFree(g->fix); cudaFree(g->stage);
  if (g->sc_host) cudaFreeHost(g->sc_host);
  if (g->pev) { for (int e = 0; e < 2 * KH_PROF_POOL; e++) if (g->pev[e]) cudaEventDestroy(g->pev[e]); delete[] g->pev; }
  delete[] g->pkind;
  for (int s = 0; s < 2; s++) { if (g->side[s]) cudaStreamDestroy(g->side[s]); if (g->ev_join[s]) cudaEventDestroy(g->ev_join[s]); }
  if (g->ev_fork) cudaEventDestroy(g->ev_fork);
  if (g->own_stream) cudaStreamDestroy(g->stream);
  delete g;
  return KH_OK;
}

int kh_grid_create(const kh_params* p, void* cuda_stream, kh_grid** out) {
  if (!p || !out) return KH_EINVAL;
  if (p->n1 < 1 || p->n2 < 1 || p->n3 < 1) return KH_EINVAL;
  if (p->coords < 0 || p->coords > 2 || p->recon < 0 || p->recon > 1 || p->inverter < 0 || p->inverter > 1 || p->fofc < 0 || p->fofc > 1 || p->floor_frame < 0 || p->floor_frame > 2 || p->transport < 0 || p->transport > 1 || p->emf < 0 || p->emf > 2) return KH_EINVAL;
  if (!(p->gamma > 1.0) || !(p->cfl > 0.0) || !(p->dt_growth_max > 0.0)) return KH_EINVAL;
  const int N[3] = {p->n1, p->n2, p->n3};
  for (int d = 0; d < 3; d++) {
    if (!(p->xmax[d] > p->xmin[d])) return KH_EINVAL;
    for (int s = 0; s < 2; s++) {
      int bc = p->bc[2 * d + s];
      if (bc < 0 || bc > 4) return KH_EINVAL;
      if (bc == KH_BC_POLAR && (d != 1 || N[d] < KH_NGH)) return KH_EINVAL;
      if (bc == KH_BC_BLOCK && (N[d] < KH_NGH || p->fofc || p->transport != KH_B_FLUX_CT || p->emf != KH_EMF_ARITHMETIC)) return KH_EINVAL;
    }
    if ((p->bc[2 * d] == KH_BC_PERIODIC) != (p->bc[2 * d + 1] == KH_BC_PERIODIC)) return KH_EINVAL;
  }
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (ndev < 1) { snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device"); return KH_ECUDA; }

  kh_grid* g = new (std::nothrow) kh_grid;
  if (!g) return KH_ENOMEM;
  memset(g, 0, sizeof(*g));
  g->p = *p;
  g->stream = (cudaStream_t)cuda_stream;
  if (!g->stream) {
    // The legacy default stream cannot be captured into a CUDA graph: use an own BLOCKING stream, which
    // still orders against work the caller enqueues on the legacy default stream.
    if (cudaStreamCreateWithFlags(&g->stream, cudaStreamDefault) != cudaSuccess) { delete g; return KH_ECUDA; }
    g->own_stream = true;
  }
  g->flat = (p->coords == KH_MINKOWSKI);
  for (int b = 0; b < 6; b++) { g->has_fixed = g->has_fixed || p->bc[b] == KH_BC_FIXED; g->has_block = g->has_block || p->bc[b] == KH_BC_BLOCK; }
  {
    int dev = 0;
    cudaGetDevice(&dev);
    g->device = dev;
    cudaDeviceGetAttribute(&g->sm_count, cudaDevAttrMultiProcessorCount, dev);
    setup_march_kernels();
    int nb = 0;
    const bool w5 = p->recon == KH_RECON_WENO5;
    const size_t smem = w5 ? MarchRing<1>::BYTES : MarchRing<0>::BYTES;
    cudaError_t eo;
    if (g->flat) eo = w5 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, flux_march_kernel<2, 1, true>, 128, smem)
                         : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, flux_march_kernel<2, 0, true>, 128, smem);
    else eo = w5 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, flux_march_kernel<2, 1, false>, 128, smem)
                 : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, flux_march_kernel<2, 0, false>, 128, smem);
    g->flux_blocks_per_sm = (eo == cudaSuccess && nb > 0) ? nb : 3;
    if (g->sm_count < 1) g->sm_count = 148;
  }
  g->use_graph = true;
  g->flux_concurrent = true;
  for (int s = 0; s < 2; s++) {
    if (cudaStreamCreateWithFlags(&g->side[s], cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&g->ev_join[s], cudaEventDisableTiming) != cudaSuccess) { kh_grid_destroy(g); return KH_ECUDA; }
  }
  if (cudaEventCreateWithFlags(&g->ev_fork, cudaEventDisableTiming) != cudaSuccess) { kh_grid_destroy(g); return KH_ECUDA; }
  g->update_tma = (p->n1 % 2 == 0);
  if (const char* e = getenv("KH_UPDATE_TMA")) g->update_tma = g->update_tma && atoi(e) != 0;
  if (g->update_tma) {
    // (the maps themselves are encoded after the allocations below)
    // the FOFC pass and the face-CT flag select the MODE at launch: set up every instantiation this grid can launch
    for (int face = 0; face < 2; face++) {
      if (face && p->transport != KH_B_FACE_CT) continue;
      if (setup_update_tma(g->flat, p->inverter + 2 * p->floor_frame + (face ? 8 : 0)) != cudaSuccess) g->update_tma = false;
    }
    cudaGetLastError();
  }
  // A/B switches for measurements (profiles/): the defaults are the product path
  if (const char* e = getenv("KH_FLUX_CONCURRENT")) g->flux_concurrent = atoi(e) != 0;
  if (const char* e = getenv("KH_MARCH_J")) g->march_J = atoi(e);
  GV& v = g->gv;
  v.n1 = p->n1; v.n2 = p->n2; v.n3 = p->n3;
  v.nt1 = v.n1 + 2 * KH_NGH; v.nt2 = v.n2 + 2 * KH_NGH; v.nt3 = v.n3 + 2 * KH_NGH;
  v.s2 = v.nt1; v.s3 = (long)v.nt1 * v.nt2; v.ntot = v.s3 * v.nt3;
  v.n2d = (long)v.nt1 * v.nt2;
  // zone numbers are held in 32 bits in several kernels (failure list, fill and update tile indices); 8 x ntot doubles of one
  // state array beyond that would not fit the device anyway
  if (v.ntot >= (1L << 31)) { kh_grid_destroy(g); return KH_EINVAL; }
  v.idx1 = v.n1 / (p->xmax[0] - p->xmin[0]); v.idx2 = v.n2 / (p->xmax[1] - p->xmin[1]); v.idx3 = v.n3 / (p->xmax[2] - p->xmin[2]);
  v.gam = p->gamma;
  for (int b = 0; b < 6; b++) v.bc[b] = p->bc[b];
  v.polar_lo = p->bc[2] == KH_BC_POLAR; v.polar_hi = p->bc[3] == KH_BC_POLAR;
  v.ndim_mask = (v.n1 > 1 ? 1 : 0) | (v.n2 > 1 ? 2 : 0) | (v.n3 > 1 ? 4 : 0);
  {
    // transverse ghost rows of the face fluxes that nothing reads (GV): only with the arithmetic EMFs and without FOFC (the other
    // EMF kernels and the re-flux read the ghost rows directly)
    const bool skip = p->emf == KH_EMF_ARITHMETIC && !p->fofc;
    v.alias2 = skip && p->bc[2] == KH_BC_PERIODIC && g->flat;
    v.alias3 = skip && p->bc[4] == KH_BC_PERIODIC;
    v.tlo2 = (v.alias2 || (skip && v.polar_lo)) ? 0 : -1;
    v.thi2 = (v.alias2 || (skip && v.polar_hi)) ? v.n2 : v.n2 + 1;
    v.tlo3 = v.alias3 ? 0 : -1;
    v.thi3 = v.alias3 ? v.n3 : v.n3 + 1;
  }
  v.fp.inv_bsq_over_rho_max = 1.0 / p->bsq_over_rho_max; v.fp.inv_bsq_over_u_max = 1.0 / p->bsq_over_u_max;
  v.fp.u_over_rho_max = p->u_over_rho_max; v.fp.gamma_max = p->gamma_max;
  v.floor_frame = p->floor_frame; v.inverter = p->inverter;

#define ALLOC(ptr, bytes)                                                       \
  do {                                                                          \
    cudaError_t e_ = cudaMalloc((void**)&(ptr), (bytes));                       \
    if (e_ != cudaSuccess) { snprintf(g_cuda_err, sizeof(g_cuda_err), "%s (alloc %zu B)", cudaGetErrorString(e_), (size_t)(bytes)); kh_grid_destroy(g); return e_ == cudaErrorMemoryAllocation ? KH_ENOMEM : KH_ECUDA; } \
    e_ = cudaMemsetAsync((ptr), 0, (bytes), g->stream);                         \
    if (e_ != cudaSuccess) { kh_grid_destroy(g); return KH_ECUDA; }             \
  } while (0)
#define ALLOC_SHIFTED(ptr, bytes)                                               \
  do {                                                                          \
    double* raw_ = nullptr;                                                     \
    ALLOC(raw_, (bytes) + 16);                                                  \
    (ptr) = raw_ + 1;                                                           \
  } while (0)
  const size_t fb = sizeof(double) * v.ntot;
  // the tables the update kernel stages by tensor copies are shifted like the zone arrays (the copy of a row starts at zone i0)
  ALLOC_SHIFTED(g->geom[0], sizeof(double) * KH_NGEO * v.n2d);
  for (int l = 1; l < 4; l++) ALLOC(g->geom[l], sizeof(double) * KH_NGEO * v.n2d);
  ALLOC(g->conn, sizeof(double) * KH_NCONN * v.n2d);
  ALLOC_SHIFTED(g->dg, sizeof(double) * KH_NDG * v.n2d);
  ALLOC_SHIFTED(g->floorp, sizeof(double) * 2 * v.n2d);
  for (int b = 0; b < 3; b++) {
    ALLOC_SHIFTED(g->P[b], KH_NP * fb);
    ALLOC_SHIFTED(g->F[b], KH_NP * fb);
    ALLOC_SHIFTED(g->ctop[b], fb);
    ALLOC_SHIFTED(g->emf[b], fb);
  }
  ALLOC(g->fix, 5 * fb);
  ALLOC(g->pflag, v.ntot);
  ALLOC(g->fflag, v.ntot);
  if (p->fofc) ALLOC(g->mask, v.ntot);
  if (p->transport == KH_B_FACE_CT) for (int b = 0; b < 3; b++) for (int d = 0; d < 3; d++) ALLOC_SHIFTED(g->Bf[b][d], fb);
  if (p->emf != KH_EMF_ARITHMETIC) for (int d = 0; d < 4; d++) ALLOC(g->ecent[d], fb);
  ALLOC(g->faillist, sizeof(unsigned) * (size_t)v.n1 * v.n2 * v.n3);
  ALLOC(g->sc, sizeof(StepScalars));
#undef ALLOC_SHIFTED
#undef ALLOC
  if (cudaMallocHost((void**)&g->sc_host, sizeof(StepScalars)) != cudaSuccess) { kh_grid_destroy(g); return KH_ENOMEM; }
  memset(g->sc_host, 0, sizeof(StepScalars));
  if (cudaMemcpyAsync(g->sc, g->sc_host, sizeof(StepScalars), cudaMemcpyHostToDevice, g->stream) != cudaSuccess) { kh_grid_destroy(g); return KH_ECUDA; }
  for (int l = 0; l < 4; l++) v.geom[l] = g->geom[l];
  v.conn = g->conn; v.dg = g->dg; v.floorp = g->floorp;
  if (g->update_tma && !make_tile_maps(g)) g->update_tma = false;      // no tensor maps: the per-thread update kernel

  GeomPar gp;
  gp.coords = p->coords; gp.a = p->a; gp.hslope = p->hslope; gp.poly_xt = p->poly_xt; gp.poly_alpha = p->poly_alpha;
  gp.mks_smooth = p->mks_smooth; gp.x1_start = p->xmin[0];
  gp.xmin1 = p->xmin[0]; gp.xmin2 = p->xmin[1];
  gp.dx1 = (p->xmax[0] - p->xmin[0]) / v.n1; gp.dx2 = (p->xmax[1] - p->xmin[1]) / v.n2;
  gp.nt1 = v.nt1; gp.nt2 = v.nt2; gp.n2 = v.n2; gp.polar_lo = v.polar_lo; gp.polar_hi = v.polar_hi;
  gp.rho_min = p->rho_min; gp.u_min = p->u_min; gp.r_char = p->r_char; gp.gamma = p->gamma;
  geometry_kernel<<<dim3((v.nt1 + 63) / 64, v.nt2), 64, 0, g->stream>>>(gp, g->geom[0], g->geom[1], g->geom[2], g->geom[3], g->conn, g->dg, g->floorp);
  g->launches++;
  cudaError_t e = cudaStreamSynchronize(g->stream);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) { snprintf(g_cuda_err, sizeof(g_cuda_err), "%s (geometry)", cudaGetErrorString(e)); kh_grid_destroy(g); return KH_ECUDA; }
  *out = g;
  return KH_OK;
}

// copy helper: device<->caller buffer, host buffers synchronise
static int xfer(kh_grid* g, void* dst, const void* src, size_t bytes, int mem, bool to_caller) {
  cudaMemcpyKind kind = (mem == KH_MEM_HOST) ? (to_caller ? cudaMemcpyDeviceToHost : cudaMemcpyHostToDevice) : cudaMemcpyDeviceToDevice;
  CK(cudaMemcpyAsync(dst, src, bytes, kind, g->stream));
  if (mem == KH_MEM_HOST) CK(cudaStreamSynchronize(g->stream));
  return KH_OK;
}

int kh_set_prims(kh_grid* g, const double* p, int with_ghosts, int mem) {
  if (!g || !p || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  if (g->has_fixed && !with_ghosts && !g->fixed_ghosts_set) return KH_EINVAL;   // FIXED ghosts come from a with_ghosts = 1 load
  ENTER(g);
  const GV& v = g->gv;
  double* Pn = g->P[g->cur];
  int rc;
  if (with_ghosts) {
    rc = xfer(g, Pn, p, sizeof(double) * KH_NP * v.ntot, mem, false);
    if (rc) return rc;
    g->fixed_ghosts_set = true;
  } else {
    size_t bytes = sizeof(double) * KH_NP * (size_t)v.n1 * v.n2 * v.n3;
    const double* src = p;
    if (mem == KH_MEM_HOST) {
      rc = ensure_stage(g);
      if (rc) return rc;
      rc = xfer(g, g->stage, p, bytes, mem, false);
      if (rc) return rc;
      src = g->stage;
    }
    pack_interior_kernel<<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, src, Pn, 1, KH_NP);
    g->launches++;
    CK(cudaGetLastError());
  }
  if (g->p.transport == KH_B_FACE_CT && g->faces_set) {
    // the face field is the magnetic state: the zone-centred B of the new primitives is slaved to it again
    double* const* B = g->Bf[g->cur];
    face_to_cent_kernel<<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, B[0], B[1], B[2], Pn, g->flat ? 1 : 0);
    g->launches++;
    CK(cudaGetLastError());
  }
  rc = fill_ghosts(g, Pn, nullptr);
  if (rc) return rc;
  if (with_ghosts && g->has_fixed) {
    // FIXED ghost layers, and the ghost zones filled FROM them (edges and corners shared with another boundary), must exist in
    // every rotating buffer: during a step only the images of interior zones are rewritten
    for (int b = 1; b < 3; b++) CK(cudaMemcpyAsync(g->P[(g->cur + b) % 3], Pn, sizeof(double) * KH_NP * v.ntot, cudaMemcpyDeviceToDevice, g->stream));
  }
  if (mem == KH_MEM_HOST) CK(cudaStreamSynchronize(g->stream));
  return KH_OK;
}

int kh_get_prims(kh_grid* g, double* p, int with_ghosts, int mem) {
  if (!g || !p || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  ENTER(g);
  const GV& v = g->gv;
  if (with_ghosts) return xfer(g, p, g->P[g->cur], sizeof(double) * KH_NP * v.ntot, mem, true);
  size_t bytes = sizeof(double) * KH_NP * (size_t)v.n1 * v.n2 * v.n3;
  if (mem == KH_MEM_HOST) { int rc = ensure_stage(g); if (rc) return rc; }
  double* dst = (mem == KH_MEM_HOST) ? g->stage : p;
  pack_interior_kernel<<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, g->P[g->cur], dst, 0, KH_NP);
  g->launches++;
  CK(cudaGetLastError());
  if (mem == KH_MEM_HOST) return xfer(g, p, dst, bytes, mem, true);
  return KH_OK;
}

int kh_get_cons(kh_grid* g, double* u, int mem) {
  if (!g || !u || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  ENTER(g);
  const GV& v = g->gv;
  size_t bytes = sizeof(double) * KH_NP * (size_t)v.n1 * v.n2 * v.n3;
  if (mem == KH_MEM_HOST) { int rc = ensure_stage(g); if (rc) return rc; }
  double* dst = (mem == KH_MEM_HOST) ? g->stage : u;
  if (g->flat) cons_kernel<true><<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, g->P[g->cur], dst);
  else cons_kernel<false><<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, g->P[g->cur], dst);
  g->launches++;
  CK(cudaGetLastError());
  if (mem == KH_MEM_HOST) return xfer(g, u, dst, bytes, mem, true);
  return KH_OK;
}

int kh_get_flags(kh_grid* g, int* pflag, int* fflag, int mem) {
  if (!g || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  ENTER(g);
  const GV& v = g->gv;
  size_t nin = (size_t)v.n1 * v.n2 * v.n3;
  int* outs[2] = {pflag, fflag};
  unsigned char* srcs[2] = {g->pflag, g->fflag};
  for (int a = 0; a < 2; a++) {
    if (!outs[a]) continue;
    if (mem == KH_MEM_HOST) { int rc = ensure_stage(g); if (rc) return rc; }
    int* dst = (mem == KH_MEM_HOST) ? (int*)g->stage : outs[a];
    flags_to_int_kernel<<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, srcs[a], dst);
    g->launches++;
    CK(cudaGetLastError());
    if (mem == KH_MEM_HOST) { int rc = xfer(g, outs[a], dst, sizeof(int) * nin, mem, true); if (rc) return rc; }
  }
  return KH_OK;
}

static int read_scalars(kh_grid* g) {
  CK(cudaMemcpyAsync(g->sc_host, g->sc, sizeof(StepScalars), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return KH_OK;
}

int kh_estimate_dt(kh_grid* g, double* dt) {
  if (!g || !dt) return KH_EINVAL;
  ENTER(g);
  const GV& v = g->gv;
  if (g->flat) estimate_dt_kernel<true><<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, g->P[g->cur], g->sc);
  else estimate_dt_kernel<false><<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, g->P[g->cur], g->sc);
  g->launches++;
  CK(cudaGetLastError());
  int rc = read_scalars(g);
  if (rc) return rc;
  double rate;
  memcpy(&rate, &g->sc_host->rate_bits, sizeof(double));
  CK(cudaMemsetAsync(&g->sc->rate_bits, 0, sizeof(unsigned long long), g->stream));
  CK(cudaStreamSynchronize(g->stream));
  if (g->sc_host->nonfinite) {               // a non-finite wave speed (fmax would have dropped it from the maximum)
    CK(cudaMemsetAsync(&g->sc->nonfinite, 0, sizeof(unsigned long long), g->stream));
    return KH_ENAN;
  }
  if (!(rate > 0.0)) return KH_ENAN;
  *dt = g->p.cfl * (1.0 / rate);            // min over zones of 1/rate = 1/max rate
  return KH_OK;
}

int kh_step(kh_grid* g, double dt, double* dt_next) {
  if (!g || dt != dt) return KH_EINVAL;
  if (g->p.transport == KH_B_FACE_CT && !g->faces_set) return KH_EINVAL;   // the face field is the magnetic state: set it first
  if (g->has_fixed && !g->fixed_ghosts_set) return KH_EINVAL;               // FIXED ghost layers were never supplied
  if (g->has_block) return KH_EINVAL;                                       // a block with KH_BC_BLOCK sides steps with its neighbours: kh_step_blocks
  if (!(dt > 0.0) && !g->have_dt_next) return KH_EINVAL;                    // no dt_next on the device yet
  ENTER(g);
  NvtxRange range_("kh_step");
  set_dt_kernel<<<1, 1, 0, g->stream>>>(g->sc, dt, dt > 0.0 ? 0 : 1);
  g->launches++;
  CK(cudaGetLastError());
  int cur = g->cur;
  bool replayed = false;
  if (g->use_graph) {
    cudaGraphExec_t* slot = g->profile ? &g->gexec_prof[cur] : &g->gexec[cur];
    if (!*slot) {
      // Capture one step.  Any failure (a stream that cannot be captured, a capture already active on it, ...) switches
      // this grid to direct launches for good: the same kernels, enqueued one by one.
      const long long before = g->launches;
      cudaGraph_t graph = nullptr;
      cudaError_t e = cudaStreamBeginCapture(g->stream, cudaStreamCaptureModeThreadLocal);
      int rc = KH_OK;
      if (e == cudaSuccess) {
        if (g->profile) { g->gp_capture = cur + 1; g->gpn[cur] = 0; }
        rc = enqueue_step(g, cur);
        g->gp_capture = 0;
        e = cudaStreamEndCapture(g->stream, &graph);
        g->graph_launches = g->launches - before;
        g->launches = before;
        if (e == cudaSuccess && rc == KH_OK) e = cudaGraphInstantiate(slot, graph, 0);
        if (graph) cudaGraphDestroy(graph);
      }
      if (e != cudaSuccess || rc != KH_OK) {
        cudaGetLastError();
        if (*slot) { cudaGraphExecDestroy(*slot); *slot = nullptr; }
        g->use_graph = false;
      }
    }
    if (*slot) {
      CK(cudaGraphLaunch(*slot, g->stream));
      g->launches += g->graph_launches;
      replayed = true;
      if (g->profile) {           // read the event nodes of this replay out before the next one overwrites them
        CK(cudaStreamSynchronize(g->stream));
        for (int r = 0; r < g->gpn[cur]; r++) {
          float ms = 0.f;
          if (cudaEventElapsedTime(&ms, g->gpev[cur][r][0], g->gpev[cur][r][1]) == cudaSuccess) {
            g->prof_ms[g->gpkind[cur][r]] += ms;
            g->prof_n[g->gpkind[cur][r]]++;
          }
        }
      }
    }
  }
  if (!replayed) {
    int rc = enqueue_step(g, cur);
    if (rc) return rc;
  }
  g->cur = (cur + 2) % 3;
  g->have_dt_next = true;
  if (dt_next) {
    int rc = read_scalars(g);
    if (rc) return rc;
    if (g->sc_host->nonfinite || !(g->sc_host->dt_next == g->sc_host->dt_next)) return KH_ENAN;   // a non-finite wave speed reached the CFL reduction
    *dt_next = g->sc_host->dt_next;
  }
  return KH_OK;
}

int kh_get_stream(kh_grid* g, void** cuda_stream) {
  if (!g || !cuda_stream) return KH_EINVAL;
  *cuda_stream = (void*)g->stream;
  return KH_OK;
}

int kh_sync(kh_grid* g) {
  if (!g) return KH_EINVAL;
  ENTER(g);
  CK(cudaStreamSynchronize(g->stream));
  return KH_OK;
}

// ---- several blocks on one device ----
static long halo_count(const GV& v, int dir) {
  const long e1 = dir == 1 ? v.nt2 : v.nt1, e2 = dir == 3 ? v.nt2 : v.nt3;
  return (long)KH_NGH * e1 * e2;
}

int kh_link_blocks(kh_grid* lo, kh_grid* hi, int dir) {
  if (!lo || !hi || dir < 1 || dir > 3) return KH_EINVAL;
  const int d = dir - 1;
  if (lo->p.bc[2 * d + 1] != KH_BC_BLOCK || hi->p.bc[2 * d] != KH_BC_BLOCK) return KH_EINVAL;
  if (lo->stream != hi->stream || lo->device != hi->device) return KH_EINVAL;
  const int nl[3] = {lo->p.n1, lo->p.n2, lo->p.n3}, nh[3] = {hi->p.n1, hi->p.n2, hi->p.n3};
  for (int e = 0; e < 3; e++) {
    if (e != d && nl[e] != nh[e]) return KH_EINVAL;                                             // same transverse shape
    const double dl = (lo->p.xmax[e] - lo->p.xmin[e]) / nl[e], dh = (hi->p.xmax[e] - hi->p.xmin[e]) / nh[e];
    if (!(fabs(dl - dh) <= 1e-12 * fabs(dl))) return KH_EINVAL;                                 // same zone size
  }
  if (lo->p.coords != hi->p.coords || lo->p.recon != hi->p.recon || lo->p.inverter != hi->p.inverter || lo->p.floor_frame != hi->p.floor_frame ||
      lo->p.gamma != hi->p.gamma || lo->p.cfl != hi->p.cfl) return KH_EINVAL;
  ENTER(lo);
  const size_t bytes = sizeof(double) * (KH_NP + 1) * (size_t)halo_count(lo->gv, dir);
  if (!lo->halo_buf[d][1]) CK(cudaMalloc((void**)&lo->halo_buf[d][1], bytes));
  if (!hi->halo_buf[d][0]) CK(cudaMalloc((void**)&hi->halo_buf[d][0], bytes));
  lo->nb[d][1] = hi;
  hi->nb[d][0] = lo;
  return KH_OK;
}

// every linked side: pack the sender's 3 layers, then unpack into the receiver's ghosts (all packs first: a block thinner than
// 6 zones would otherwise send layers its own unpack has just overwritten -- not possible here, ghosts are not interior, but
// the order also is what a two-sided transport needs)
static int exchange(kh_grid* const* blocks, int n, int which /* offset of the P buffer from cur */) {
  for (int pass = 0; pass < 2; pass++)
    for (int b = 0; b < n; b++) {
      kh_grid* g = blocks[b];
      for (int d = 0; d < 3; d++) for (int sd = 0; sd < 2; sd++) {
        if (g->p.bc[2 * d + sd] != KH_BC_BLOCK) continue;
        kh_grid* nbr = g->nb[d][sd];
        if (!nbr) return KH_EINVAL;                                                              // a KH_BC_BLOCK side that was never linked
        const long cnt = halo_count(g->gv, d + 1);
        const unsigned grid = (unsigned)((cnt + 127) / 128);
        if (pass == 0) halo_pack_kernel<<<grid, 128, 0, g->stream>>>(g->gv, g->P[(g->cur + which) % 3], g->pflag, d + 1, sd, g->halo_buf[d][sd]);
        else halo_unpack_kernel<<<grid, 128, 0, g->stream>>>(g->gv, g->P[(g->cur + which) % 3], g->pflag, d + 1, sd, nbr->halo_buf[d][1 - sd]);
        g->launches++;
      }
    }
  CK(cudaGetLastError());
  return KH_OK;
}

static int check_blocks(kh_grid* const* blocks, int n) {
  if (!blocks || n < 1 || n > 16) return KH_EINVAL;
  for (int b = 0; b < n; b++) {
    if (!blocks[b] || blocks[b]->stream != blocks[0]->stream || blocks[b]->cur != blocks[0]->cur) return KH_EINVAL;
    if (blocks[b]->has_fixed && !blocks[b]->fixed_ghosts_set) return KH_EINVAL;
  }
  return KH_OK;
}

int kh_exchange_halos(kh_grid* const* blocks, int n) {
  int rc = check_blocks(blocks, n);
  if (rc) return rc;
  ENTER(blocks[0]);
  return exchange(blocks, n, 0);
}

int kh_step_blocks(kh_grid* const* blocks, int n, double dt, double* dt_next) {
  int rc = check_blocks(blocks, n);
  if (rc) return rc;
  if (dt != dt) return KH_EINVAL;
  for (int b = 0; b < n; b++) if (!(dt > 0.0) && !blocks[b]->have_dt_next) return KH_EINVAL;
  ENTER(blocks[0]);
  for (int b = 0; b < n; b++) {
    kh_grid* g = blocks[b];
    set_dt_kernel<<<1, 1, 0, g->stream>>>(g->sc, dt, dt > 0.0 ? 0 : 1);
    g->launches++;
  }
  const int cur = blocks[0]->cur;
  for (int sub = 0; sub < 2; sub++) {
    const int out = sub == 0 ? 1 : 2;                      // P* = P[cur + 1], P^{n+1} = P[cur + 2]
    for (int b = 0; b < n; b++) {                          // K2, K3, K4/K5 and the block's own boundary fills
      kh_grid* g = blocks[b];
      rc = substep(g, g->P[cur], sub == 0 ? g->P[cur] : g->P[(cur + 1) % 3], g->P[(cur + out) % 3], sub == 0 ? 0.5 : 1.0, sub == 1,
                   nullptr, nullptr, false);
      if (rc) return rc;
    }
    rc = exchange(blocks, n, out);                         // first synchronisation: primitives and inversion flags
    if (rc) return rc;
    for (int b = 0; b < n; b++) {                          // K5b: failed zones read their neighbours through the halo
      rc = do_fixup(blocks[b], blocks[b]->P[(cur + out) % 3]);
      if (rc) return rc;
    }
    rc = exchange(blocks, n, out);                         // second synchronisation: the repaired zones reach the neighbours' ghosts
    if (rc) return rc;
  }
  BlockScalars bs;
  bs.n = n;
  for (int b = 0; b < n; b++) bs.sc[b] = blocks[b]->sc;
  finalize_dt_blocks_kernel<<<1, 1, 0, blocks[0]->stream>>>(bs, blocks[0]->p.cfl, blocks[0]->p.dt_growth_max);
  blocks[0]->launches++;
  CK(cudaGetLastError());
  for (int b = 0; b < n; b++) { blocks[b]->cur = (cur + 2) % 3; blocks[b]->have_dt_next = true; }
  if (dt_next) {
    rc = read_scalars(blocks[0]);
    if (rc) return rc;
    if (blocks[0]->sc_host->nonfinite || !(blocks[0]->sc_host->dt_next == blocks[0]->sc_host->dt_next)) return KH_ENAN;
    *dt_next = blocks[0]->sc_host->dt_next;
  }
  return KH_OK;
}

int kh_divB(kh_grid* g, double* max_abs) {
  if (!g || !max_abs) return KH_EINVAL;
  ENTER(g);
  const GV& v = g->gv;
  int lo[3], cnt[3];
  const int N[3] = {v.n1, v.n2, v.n3};
  // corners on a lower boundary plane involve ghost zones: valid where those are periodic images or a neighbouring block's zones
  for (int d = 0; d < 3; d++) { lo[d] = (g->p.bc[2 * d] == KH_BC_PERIODIC || g->p.bc[2 * d] == KH_BC_BLOCK) ? 0 : 1; cnt[d] = N[d] - lo[d]; }
  unsigned long long zero = 0;
  CK(cudaMemcpyAsync(&g->sc->max_bits, &zero, sizeof(zero), cudaMemcpyHostToDevice, g->stream));
  if (cnt[0] > 0 && cnt[1] > 0 && cnt[2] > 0) {
    divb_kernel<<<zone_grid(cnt[0], cnt[1], cnt[2]), 128, 0, g->stream>>>(v, g->P[g->cur], g->sc, lo[0], lo[1], lo[2]);
    g->launches++;
    CK(cudaGetLastError());
  }
  int rc = read_scalars(g);
  if (rc) return rc;
  memcpy(max_abs, &g->sc_host->max_bits, sizeof(double));
  return KH_OK;
}

int kh_set_face_B(kh_grid* g, const double* f1, const double* f2, const double* f3, int mem) {
  if (!g || !f1 || !f2 || !f3 || g->p.transport != KH_B_FACE_CT || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  const GV& v = g->gv;
  const double* f[3] = {f1, f2, f3};
  for (int d = 0; d < 3; d++) {
    int rc = xfer(g, g->Bf[g->cur][d], f[d], sizeof(double) * v.ntot, mem, false);
    if (rc) return rc;
  }
  double* const* B = g->Bf[g->cur];
  face_to_cent_kernel<<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, B[0], B[1], B[2], g->P[g->cur], g->flat ? 1 : 0);
  g->launches++;
  CK(cudaGetLastError());
  int rc = fill_ghosts(g, g->P[g->cur], nullptr);
  if (rc) return rc;
  CK(cudaStreamSynchronize(g->stream));
  g->faces_set = true;
  return KH_OK;
}

int kh_get_face_B(kh_grid* g, double* f1, double* f2, double* f3, int mem) {
  if (!g || !f1 || !f2 || !f3 || g->p.transport != KH_B_FACE_CT || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  double* f[3] = {f1, f2, f3};
  for (int d = 0; d < 3; d++) {
    int rc = xfer(g, f[d], g->Bf[g->cur][d], sizeof(double) * g->gv.ntot, mem, true);
    if (rc) return rc;
  }
  return KH_OK;
}

int kh_divB_face(kh_grid* g, double* max_abs) {
  if (!g || !max_abs || g->p.transport != KH_B_FACE_CT) return KH_EINVAL;
  const GV& v = g->gv;
  unsigned long long zero = 0;
  CK(cudaMemcpyAsync(&g->sc->max_bits, &zero, sizeof(zero), cudaMemcpyHostToDevice, g->stream));
  double* const* B = g->Bf[g->cur];
  divb_face_kernel<<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, B[0], B[1], B[2], g->sc);
  g->launches++;
  CK(cudaGetLastError());
  int rc = read_scalars(g);
  if (rc) return rc;
  long long bits = (long long)g->sc_host->max_bits;
  double val;
  memcpy(&val, &bits, sizeof(val));
  *max_abs = val;
  return KH_OK;
}

int kh_count_flags(kh_grid* g, long long* n_pflag, long long* n_fflag) {
  if (!g) return KH_EINVAL;
  ENTER(g);
  int rc = read_scalars(g);
  if (rc) return rc;
  if (n_pflag) *n_pflag = (long long)g->sc_host->n_pflag;
  if (n_fflag) *n_fflag = (long long)g->sc_host->n_fflag;
  return KH_OK;
}

int kh_get_geom(kh_grid* g, int loc, double* gcov16, double* gcon16, double* gdet, double* alpha, int mem) {
  if (!g || loc < 0 || loc > 3 || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  const long n2d = g->gv.n2d;
  double *d_cov = gcov16, *d_con = gcon16, *d_det = gdet, *d_al = alpha;
  if (mem == KH_MEM_HOST) {
    int rc = ensure_stage(g);
    if (rc) return rc;
    double* s = g->stage;   // >= 64 * n2d doubles
    d_cov = gcov16 ? s : nullptr; d_con = gcon16 ? s + 16 * n2d : nullptr; d_det = gdet ? s + 32 * n2d : nullptr; d_al = alpha ? s + 33 * n2d : nullptr;
  }
  geom_export_kernel<<<(unsigned)((n2d + 127) / 128), 128, 0, g->stream>>>(n2d, g->geom[loc], d_cov, d_con, d_det, d_al);
  g->launches++;
  CK(cudaGetLastError());
  if (mem == KH_MEM_HOST) {
    if (gcov16) CK(cudaMemcpyAsync(gcov16, d_cov, sizeof(double) * 16 * n2d, cudaMemcpyDeviceToHost, g->stream));
    if (gcon16) CK(cudaMemcpyAsync(gcon16, d_con, sizeof(double) * 16 * n2d, cudaMemcpyDeviceToHost, g->stream));
    if (gdet) CK(cudaMemcpyAsync(gdet, d_det, sizeof(double) * n2d, cudaMemcpyDeviceToHost, g->stream));
    if (alpha) CK(cudaMemcpyAsync(alpha, d_al, sizeof(double) * n2d, cudaMemcpyDeviceToHost, g->stream));
    CK(cudaStreamSynchronize(g->stream));
  }
  return KH_OK;
}

int kh_get_conn(kh_grid* g, double* conn64, int mem) {
  if (!g || !conn64 || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  const long n2d = g->gv.n2d;
  if (mem == KH_MEM_HOST) { int rc = ensure_stage(g); if (rc) return rc; }
  double* dst = (mem == KH_MEM_HOST) ? g->stage : conn64;
  conn_export_kernel<<<(unsigned)((n2d + 127) / 128), 128, 0, g->stream>>>(n2d, g->conn, dst);
  g->launches++;
  CK(cudaGetLastError());
  if (mem == KH_MEM_HOST) return xfer(g, conn64, dst, sizeof(double) * 64 * n2d, mem, true);
  return KH_OK;
}

int kh_get_flux(kh_grid* g, int dir, double* F, double* ctop, int mem) {
  if (!g || dir < 1 || dir > 3 || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  const GV& v = g->gv;
  const size_t fb = sizeof(double) * v.ntot;
  if (F) {
    int rc = ensure_stage(g);
    if (rc) return rc;
    CK(cudaMemcpyAsync(g->stage, g->F[dir - 1], KH_NP * fb, cudaMemcpyDeviceToDevice, g->stream));
    ct_flux_debug_kernel<<<zone_grid(v.n1 + 1, v.n2 + 1, v.n3 + 1), 128, 0, g->stream>>>(v, dir, g->stage, g->emf[0], g->emf[1], g->emf[2]);
    g->launches++;
    CK(cudaGetLastError());
    rc = xfer(g, F, g->stage, KH_NP * fb, mem, true);
    if (rc) return rc;
  }
  if (ctop) return xfer(g, ctop, g->ctop[dir - 1], fb, mem, true);
  return KH_OK;
}

int kh_get_emf(kh_grid* g, int dir, double* emf, int mem) {
  if (!g || !emf || dir < 1 || dir > 3 || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  return xfer(g, emf, g->emf[dir - 1], sizeof(double) * g->gv.ntot, mem, true);
}

int kh_debug_predictor(kh_grid* g, double dt) {
  if (!g || !(dt > 0.0)) return KH_EINVAL;
  if (g->p.transport == KH_B_FACE_CT && !g->faces_set) return KH_EINVAL;
  set_dt_kernel<<<1, 1, 0, g->stream>>>(g->sc, dt, 0);
  g->launches++;
  const bool face = g->p.transport == KH_B_FACE_CT;
  int rc = substep(g, g->P[g->cur], g->P[g->cur], g->P[(g->cur + 1) % 3], 0.5, false, face ? g->Bf[g->cur] : nullptr,
                   face ? g->Bf[(g->cur + 1) % 3] : nullptr);
  if (rc) return rc;
  g->cur = (g->cur + 1) % 3;
  CK(cudaStreamSynchronize(g->stream));
  return KH_OK;
}

int kh_debug_fixup(kh_grid* g, const int* pflag_with_ghosts, int mem) {
  if (!g || !pflag_with_ghosts || (mem != KH_MEM_DEVICE && mem != KH_MEM_HOST)) return KH_EINVAL;
  const GV& v = g->gv;
  const int* src = pflag_with_ghosts;
  if (mem == KH_MEM_HOST) {
    int rc = ensure_stage(g);
    if (rc) return rc;
    rc = xfer(g, g->stage, pflag_with_ghosts, sizeof(int) * v.ntot, mem, false);
    if (rc) return rc;
    src = (const int*)g->stage;
  }
  int_to_flags_kernel<<<(unsigned)((v.ntot + 127) / 128), 128, 0, g->stream>>>(v.ntot, src, g->pflag);
  g->launches++;
  CK(cudaMemsetAsync(g->fflag, 0, v.ntot, g->stream));
  reset_counters_kernel<<<1, 1, 0, g->stream>>>(g->sc, 0);
  build_faillist_kernel<<<zone_grid(v.n1, v.n2, v.n3), 128, 0, g->stream>>>(v, g->pflag, g->faillist, g->sc);
  g->launches += 2;
  int rc = do_fixup(g, g->P[g->cur]);
  if (rc) return rc;
  CK(cudaStreamSynchronize(g->stream));
  return KH_OK;
}

long long kh_launch_count(const kh_grid* g) { return g ? g->launches : 0; }

int kh_set_graph(kh_grid* g, int enable) {
  if (!g) return KH_EINVAL;
  g->use_graph = enable != 0;
  if (!enable) destroy_graphs(g);
  return KH_OK;
}

int kh_set_profile(kh_grid* g, int enable) {
  if (!g) return KH_EINVAL;
  if (enable && !g->pev) {
    g->pev = new (std::nothrow) cudaEvent_t[2 * KH_PROF_POOL];
    g->pkind = new (std::nothrow) int[KH_PROF_POOL];
    if (!g->pev || !g->pkind) return KH_ENOMEM;
    memset(g->pev, 0, sizeof(cudaEvent_t) * 2 * KH_PROF_POOL);
    for (int e = 0; e < 2 * KH_PROF_POOL; e++) CK(cudaEventCreate(&g->pev[e]));
  }
  if (g->profile) prof_flush(g);
  g->profile = enable != 0;
  for (int k = 0; k < KH_K_COUNT; k++) { g->prof_ms[k] = 0.0; g->prof_n[k] = 0; }
  return KH_OK;
}

int kh_get_profile(kh_grid* g, double* ms, long long* count) {
  if (!g || !ms || !count) return KH_EINVAL;
  if (g->profile) prof_flush(g);
  for (int k = 0; k < KH_K_COUNT; k++) { ms[k] = g->prof_ms[k]; count[k] = g->prof_n[k]; }
  return KH_OK;
}

int kh_measure_fp64_peak(double* tflops, double* sm_mhz_est) {
  if (!tflops) return KH_EINVAL;
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int threads = 256, blocks = sms * 8, iters = 1 << 15;
  double* out = nullptr;
  CK(cudaMalloc((void**)&out, sizeof(double) * threads * blocks));
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0));
  CK(cudaEventCreate(&e1));
  dfma_peak_kernel<<<blocks, threads>>>(out, iters);   // warm-up
  double best = 0.0;
  for (int rep = 0; rep < 5; rep++) {
    CK(cudaEventRecord(e0));
    dfma_peak_kernel<<<blocks, threads>>>(out, iters);
    CK(cudaEventRecord(e1));
    CK(cudaEventSynchronize(e1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    double fl = 2.0 * 8.0 * (double)iters * threads * blocks;
    double tf = fl / (ms * 1e-3) / 1e12;
    if (tf > best) best = tf;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out);
  *tflops = best;
  if (sm_mhz_est) *sm_mhz_est = best * 1e12 / (2.0 * 64.0 * sms) / 1e6;   // assuming 64 fp64 FMA lanes per SM
  return KH_OK;
}

}  // extern "C"
