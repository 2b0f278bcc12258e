// chorus.cu -- C ABI of libchorus_b200.so (include/chorus.h): context, kernel dispatch, SSPRK driver.
// Every step of the hot path runs in the CUDA kernels of kernels_*.cuh / geometry.cuh; this file only owns device
// memory, marshals arguments and enqueues launches on the caller's stream.  No CPU fallback exists.
#include "../../include/chorus.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "basis.h"
#include "geometry.cuh"
#include "kernels_stage.cuh"
#include "peak.cuh"

using namespace chorus;

struct chorus_ctx {
  int n = 0, n2 = 0, n3 = 0, nf = 0;
  int64_t E = 0;          // elements of the local mesh: the owned ones first, then the ghosts of a partition
  int64_t E_own = 0;      // elements this context advances (= E unless chorus_set_owned made it a partition)
  cudaStream_t stream = nullptr;
  chorus_physics phys{};
  PhysD ph{};
  int num_sms = 0;
  size_t max_smem = 0;
  // mesh
  int ng = 0;
  double* d_xyz = nullptr;
  int32_t* d_nbr_elem = nullptr;
  uint8_t *d_nbr_face = nullptr, *d_nbr_orient = nullptr;
  // operators for the geometry kernel
  double *d_Gm = nullptr, *d_Dff = nullptr, *d_Efs = nullptr, *d_Dfs = nullptr;
  // geometry
  double *d_Sfl = nullptr, *d_detJ = nullptr, *d_jinv = nullptr, *d_xsol = nullptr, *d_krfl = nullptr, *d_nfc = nullptr;
  double* d_Sint = nullptr;         // S^d at the interior flux points (orders whose element kernel stages it: kSintOrder)
  // state registers (element-major) and face buffers
  double* d_U[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  int cur = 0;
  bool have_state = false;
  double* d_Qf[2] = {nullptr, nullptr};   // face traces, double-buffered: a stage reads one and emits the next state's into the other
  int qf_cur = 0;                         // which buffer holds the traces of the current state ...
  bool traces_valid = false;              // ... if any does
  double* d_Vf = nullptr;
  unsigned long long* d_ws = nullptr;
  double *d_wq = nullptr, *d_diag = nullptr;   // quadrature weights [n]; diagnostics partial sums [kDiagBlocks + 1][3]
  unsigned* d_arrivals = nullptr;   // per-SM CTA arrival counters of the main kernel
  // partition halo (chorus_halo_setup): faces whose traces / viscous fluxes go to, and come from, other partitions
  int64_t n_send = 0, n_recv = 0;
  int32_t *d_send_elem = nullptr, *d_recv_elem = nullptr;
  uint8_t *d_send_face = nullptr, *d_recv_face = nullptr;
  // split step (chorus_step_begin / chorus_stage_main / chorus_stage_face)
  double split_dt = 0.0;
  int split_nstages = 0, split_next = -1;   // next stage to run (-1: no split step in progress)
  bool split_face_pending = false;
  int split_b[5] = {0, 0, 0, 0, 0};
  StageIO pend{};
  double* d_scratch = nullptr;      // per-CTA global scratch of the scalar kernels' SPILL variants (orders 8, 9 with diffusion)
  size_t scratch_doubles = 0;
  int64_t launches = 0;
  bool use_mma = true;   // orders 4..8: two-kernel DMMA pipeline (kernels_stage.cuh); CHORUS_KERNELS=scalar selects the
                         // three-kernel shared-memory path that serves the other orders (kernels_residual.cuh)
  bool prof = false;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_ev[3];
  std::string err;
  struct HostPipe* pipe = nullptr;   // chorus_step_host: copy streams, staging buffers and events (made on first use)
};

// Pipelined host jobs (chorus_step_host): job k uses slot k % 2 of every array.
struct HostPipe {
  cudaStream_t s_in = nullptr, s_out = nullptr;          // host -> device and device -> host copies
  double* in[2] = {nullptr, nullptr};                    // staged inputs  [9][E][n3] (interface layout)
  double* out[2] = {nullptr, nullptr};                   // staged results [9][E][n3]
  unsigned long long* ws[2] = {nullptr, nullptr};        // wave speed of the result (bits of a double)
  cudaEvent_t in_ready[2] = {}, in_free[2] = {}, out_ready[2] = {}, out_free[2] = {};
  int64_t jobs = 0;
};

namespace {

constexpr int kDiagBlocks = 1184;   // 8 x 148: blocks of the diagnostics reduction (fixed, so the summation tree is too)

int fail(chorus_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
#define CU(c, call)                                                                                          \
  do {                                                                                                       \
    cudaError_t e_ = (call);                                                                                 \
    if (e_ != cudaSuccess) return fail(c, CHORUS_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
  } while (0)

struct ProfScope {   // brackets one launch with events when profiling is on
  chorus_ctx* c;
  int cls;
  cudaEvent_t a = nullptr, b = nullptr;
  ProfScope(chorus_ctx* c_, int cls_) : c(c_), cls(cls_) {
    if (c->prof && cudaEventCreate(&a) == cudaSuccess && cudaEventCreate(&b) == cudaSuccess) cudaEventRecord(a, c->stream);
  }
  ~ProfScope() {
    if (a && b) {
      cudaEventRecord(b, c->stream);
      c->prof_ev[cls].push_back({a, b});
    }
  }
};

PhysD to_device_phys(const chorus_physics& p) {
  PhysD d;
  d.gamma = p.gamma; d.gm1 = p.gamma - 1.0; d.R = p.R_gas; d.Cp = p.Cp; d.GM = p.GM; d.Omega = p.Omega;
  d.nu = p.nu; d.kappa = p.kappa; d.eta = p.eta; d.c_h = p.c_h; d.a_psi = p.a_psi; d.q_bottom = p.q_bottom; d.T_top = p.T_top;
  d.iR = 1.0 / p.R_gas; d.igamma = 1.0 / p.gamma;
  d.bc_inner = p.bc_mag_inner; d.bc_outer = p.bc_mag_outer; d.flags = p.flags;
  return d;
}

int grid_1d(const chorus_ctx* c, int64_t total, int block) {
  int64_t g = (total + block - 1) / block;
  int64_t cap = (int64_t)c->num_sms * 16;
  return (int)(g < cap ? (g < 1 ? 1 : g) : cap);
}

// which gradient the residual kernel needs
int gradv_of(const chorus_physics& p) { return (p.flags & kFlagDiffusion) ? 2 : (p.flags & kFlagPowell) ? 1 : 0; }

template <int N>
struct Hot {
  using I = Ix<N>;
  // per-CTA global scratch for the SPILL variants of the scalar kernels (orders whose tiles exceed shared memory)
  static int need_scratch(chorus_ctx* c, size_t doubles) {
    if (c->scratch_doubles >= doubles) return CHORUS_OK;
    cudaFree(c->d_scratch);
    c->d_scratch = nullptr;
    c->scratch_doubles = 0;
    CU(c, cudaMalloc(&c->d_scratch, sizeof(double) * doubles));
    c->scratch_doubles = doubles;
    return CHORUS_OK;
  }
  template <bool DIFF, int GRADV, bool SPILL>
  static int residual_launch_impl(chorus_ctx* c, const double* Qin, const StageOut& out) {
    constexpr size_t smem = residual_smem_bytes<N, DIFF, GRADV, SPILL>();
    if (smem > c->max_smem)
      return fail(c, CHORUS_EINVAL, "order " + std::to_string(N) + " with these physics flags needs " + std::to_string(smem) +
                                        " B of shared memory per CTA (limit " + std::to_string(c->max_smem) + ")");
    auto k = residual_kernel<N, DIFF, GRADV, SPILL>;
    CU(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 1;
    constexpr int threads = ScalarCfg<N>::kThreads;
    CU(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, threads, smem));
    if (occ < 1) occ = 1;
    const int64_t cap = (int64_t)c->num_sms * occ;
    const int grid = (int)(c->E < cap ? c->E : cap);
    if (SPILL) {
      int rc = need_scratch(c, residual_scratch_doubles<N, DIFF, GRADV>() * (size_t)grid);
      if (rc) return rc;
    }
    {
      ProfScope ps(c, 2);
      k<<<grid, threads, smem, c->stream>>>(c->E, c->ph, Qin, c->d_Qf[0], c->d_Vf, c->d_Sfl, c->d_detJ, c->d_jinv, c->d_xsol, c->d_krfl,
                                         c->d_nbr_elem, c->d_nbr_face, c->d_nbr_orient, out, c->d_scratch);
    }
    ++c->launches;
    CU(c, cudaGetLastError());
    return CHORUS_OK;
  }
  template <bool DIFF, int GRADV>
  static int residual_launch(chorus_ctx* c, const double* Qin, const StageOut& out) {
    if (residual_smem_bytes<N, DIFF, GRADV, false>() <= c->max_smem) return residual_launch_impl<DIFF, GRADV, false>(c, Qin, out);
    return residual_launch_impl<DIFF, GRADV, true>(c, Qin, out);
  }
  // ---- production pipeline (orders 4..8): main kernel, then (diffusion) the face kernel
  template <bool DIFF, int GRADV>
  static int main_launch(chorus_ctx* c, const StageIO& io) {
    if constexpr (kMmaOrder(N)) {
      constexpr size_t smem = stage_main_smem_bytes<N, GRADV>();
      constexpr int threads = MainCfg<N>::kThreads;
      auto k = stage_main_kernel<N, DIFF, GRADV>;
      CU(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      CU(c, cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
      int occ = 1;
      CU(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, threads, smem));
      if (occ < 1) occ = 1;
      const int64_t cap = (int64_t)c->num_sms * occ;
      const int grid = (int)(c->E_own < cap ? c->E_own : cap);
      {
        ProfScope ps(c, 2);
        k<<<grid, threads, smem, c->stream>>>(c->E_own, c->ph, io, geo(c));
      }
      ++c->launches;
      CU(c, cudaGetLastError());
      return CHORUS_OK;
    } else {
      return fail(c, CHORUS_EINVAL, "the DMMA pipeline serves orders 4..8");
    }
  }
  static int face_launch(chorus_ctx* c, const StageIO& io) {
    constexpr size_t smem = stage_face_smem_bytes<N>();
    auto k = stage_face_kernel<N>;
    CU(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 1;
    CU(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, 256, smem));
    if (occ < 1) occ = 1;
    const int64_t cap = (int64_t)c->num_sms * occ;
    const int grid = (int)(c->E_own < cap ? c->E_own : cap);
    {
      ProfScope ps(c, 1);
      k<<<grid, 256, smem, c->stream>>>(c->E_own, io, geo(c));
    }
    ++c->launches;
    CU(c, cudaGetLastError());
    return CHORUS_OK;
  }
  static Geo geo(const chorus_ctx* c) {
    return Geo{c->d_Sfl, c->d_Sint, c->d_detJ, c->d_jinv, c->d_xsol, c->d_krfl, c->d_nfc, c->d_nbr_elem, c->d_nbr_face, c->d_nbr_orient};
  }
  // one residual evaluation through the pipeline.  io carries Qe and the outputs; the traces of Qe must be in d_Qf[qf_cur].
  static int stage_pipeline_main(chorus_ctx* c, StageIO& io) {
    io.Qf = c->d_Qf[c->qf_cur];
    io.QfOut = c->d_Qf[c->qf_cur ^ 1];
    io.Vf = c->d_Vf;
    const int gv = gradv_of(c->phys);
    if (gv == 2) return main_launch<true, 2>(c, io);
    if (gv == 1) return main_launch<false, 1>(c, io);
    return main_launch<false, 0>(c, io);
  }
  static int stage_pipeline_face(chorus_ctx* c, const StageIO& io) {
    int rc = gradv_of(c->phys) == 2 ? face_launch(c, io) : CHORUS_OK;
    if (!rc && io.Qout != nullptr) c->qf_cur ^= 1;   // the traces of the new state were emitted into the other buffer
    return rc;
  }
  static int stage_pipeline(chorus_ctx* c, StageIO io) {
    int rc = stage_pipeline_main(c, io);
    return rc ? rc : stage_pipeline_face(c, io);
  }
  static int trace(chorus_ctx* c, const double* Qin, double* Qf) {
    constexpr size_t smem = sizeof(double) * 9 * I::n3;
    auto k = trace_kernel<N>;
    CU(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 1;
    CU(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, 256, smem));
    if (occ < 1) occ = 1;
    const int64_t cap = (int64_t)c->num_sms * occ;
    const int grid = (int)(c->E_own < cap ? c->E_own : cap);
    {
      ProfScope ps(c, 0);
      k<<<grid, 256, smem, c->stream>>>(c->E_own, Qin, Qf);
    }
    ++c->launches;
    CU(c, cudaGetLastError());
    return CHORUS_OK;
  }
  template <bool SPILL>
  static int grad_impl(chorus_ctx* c, const double* Qin, double* Vf, double* Gout) {
    constexpr size_t smem = grad_smem_bytes<N, SPILL>();
    if (smem > c->max_smem) return fail(c, CHORUS_EINVAL, "gradient kernel: order too high for the shared-memory budget");
    auto k = grad_kernel<N, SPILL>;
    CU(c, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 1;
    CU(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, ScalarCfg<N>::kThreads, smem));
    if (occ < 1) occ = 1;
    const int64_t cap = (int64_t)c->num_sms * occ;
    const int grid = (int)(c->E < cap ? c->E : cap);
    if (SPILL) {
      int rc = need_scratch(c, (size_t)27 * I::n3 * (size_t)grid);
      if (rc) return rc;
    }
    {
      ProfScope ps(c, 1);
      k<<<grid, ScalarCfg<N>::kThreads, smem, c->stream>>>(c->E, c->ph, Qin, c->d_Qf[0], c->d_Sfl, c->d_jinv, c->d_krfl, c->d_nbr_elem, c->d_nbr_face,
                                         c->d_nbr_orient, Vf, Gout, c->d_scratch);
    }
    ++c->launches;
    CU(c, cudaGetLastError());
    return CHORUS_OK;
  }
  static int grad(chorus_ctx* c, const double* Qin, double* Vf, double* Gout) {
    if (grad_smem_bytes<N, false>() <= c->max_smem) return grad_impl<false>(c, Qin, Vf, Gout);
    return grad_impl<true>(c, Qin, Vf, Gout);
  }
  // legacy three-kernel path (orders 2, 3, 8, 9 and CHORUS_KERNELS=scalar): trace, gradient, residual + RK
  static int stage_legacy(chorus_ctx* c, const double* Qin, const StageOut& out) {
    c->traces_valid = false;   // d_Qf[0] is this path's scratch
    c->qf_cur = 0;
    int rc = trace(c, Qin, c->d_Qf[0]);
    if (rc) return rc;
    const int gv = gradv_of(c->phys);
    if (gv == 2) {
      rc = grad(c, Qin, c->d_Vf, nullptr);
      if (rc) return rc;
      return residual_launch<true, 2>(c, Qin, out);
    }
    if (gv == 1) return residual_launch<false, 1>(c, Qin, out);
    return residual_launch<false, 0>(c, Qin, out);
  }
  // one residual evaluation of the state in Qin, fused with the output / RK combination described by `out`.
  // scratch: a state-sized buffer distinct from Qin, the outputs and the stage registers (residual mode with diffusion).
  // split: only the element kernel is launched and the stage is left pending in c->pend (chorus_stage_main); face_pending()
  // finishes it (chorus_stage_face).  A partition exchanges halo data between the two.
  static int face_pending(chorus_ctx* c) { return stage_pipeline_face(c, c->pend); }
  static int ensure_traces(chorus_ctx* c, const double* Qin) {
    if (!(c->use_mma && kMmaOrder(N))) return fail(c, CHORUS_EINVAL, "the split step serves the DMMA pipeline (orders 4..8)");
    if (!c->traces_valid) {
      int rc = trace(c, Qin, c->d_Qf[c->qf_cur]);
      if (rc) return rc;
      c->traces_valid = true;
    }
    return CHORUS_OK;
  }
  static int stage(chorus_ctx* c, const double* Qin, const StageOut& out, double* scratch, bool split = false) {
    if (!(c->use_mma && kMmaOrder(N))) return split ? fail(c, CHORUS_EINVAL, "the split step serves orders 4..8") : stage_legacy(c, Qin, out);
    if (!c->traces_valid) {
      int rc = trace(c, Qin, c->d_Qf[c->qf_cur]);
      if (rc) return rc;
      c->traces_valid = true;
    }
    StageIO io{};
    io.Qe = Qin;
    io.Rout = out.Rout;
    io.Qout = out.Qout;
    io.Part = out.Qout ? out.Qout : scratch;
    io.bdt = out.bdt;
    io.sm_arrivals = c->d_arrivals;
    {   // split the combination into the evaluated state itself (already on chip) and at most two other registers
      const double* A[3] = {out.A0, out.A1, out.A2};
      const double cc[3] = {out.c0, out.c1, out.c2};
      int k = 0;
      for (int i = 0; i < 3; ++i) {
        if (A[i] == nullptr) continue;
        if (A[i] == Qin) io.cq += cc[i];
        else if (k == 0) { io.A0 = A[i]; io.c0 = cc[i]; ++k; }
        else if (k == 1) { io.A1 = A[i]; io.c1 = cc[i]; ++k; }
        else return fail(c, CHORUS_EINVAL, "more than two foreign stage registers");
      }
    }
    if (split) {
      int rc = stage_pipeline_main(c, io);
      c->pend = io;
      return rc;
    }
    return stage_pipeline(c, io);
  }
};

// CHORUS_ONLY_ORDER=<n> (a build option of build.py, off by default) instantiates the kernels of one order only.
#ifdef CHORUS_ONLY_ORDER
#define DISPATCH_N(c, expr)                                                                  \
  [&]() -> int {                                                                             \
    if ((c)->n == CHORUS_ONLY_ORDER) { using H = Hot<CHORUS_ONLY_ORDER>; return expr; }      \
    return fail((c), CHORUS_EINVAL, "this build serves one order only (CHORUS_ONLY_ORDER)"); \
  }()
#else
#define DISPATCH_N(c, expr)                                          \
  [&]() -> int {                                                     \
    switch ((c)->n) {                                                \
      case 2: { using H = Hot<2>; return expr; }                     \
      case 3: { using H = Hot<3>; return expr; }                     \
      case 4: { using H = Hot<4>; return expr; }                     \
      case 5: { using H = Hot<5>; return expr; }                     \
      case 6: { using H = Hot<6>; return expr; }                     \
      case 7: { using H = Hot<7>; return expr; }                     \
      case 8: { using H = Hot<8>; return expr; }                     \
      case 9: { using H = Hot<9>; return expr; }                     \
      default: return fail((c), CHORUS_EINVAL, "order must be 2..9"); \
    }                                                                \
  }()
#endif

int run_geometry(chorus_ctx* c) {
  const int N1 = c->n + 1;
  const int cap = c->ng > N1 ? c->ng : N1;
  const size_t smem = sizeof(double) * 20 * (size_t)cap * cap * cap;
  if (smem > c->max_smem) return fail(c, CHORUS_EINVAL, "geometry kernel: too many geometry nodes for the shared-memory budget");
  CU(c, cudaFuncSetAttribute(geometry_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const bool need_kr = c->phys.kr_scale != 0.0;
  if (need_kr && !c->d_krfl) CU(c, cudaMalloc(&c->d_krfl, sizeof(double) * c->E * 3 * c->nf));
  if (!need_kr && c->d_krfl) {
    cudaFree(c->d_krfl);
    c->d_krfl = nullptr;
  }
  GeomOps op{c->d_Gm, c->d_Dff, c->d_Efs, c->d_Dfs};
  geometry_kernel<<<(unsigned)c->E, 256, smem, c->stream>>>(c->n, c->ng, c->E, op, c->d_xyz, c->d_Sfl, c->d_detJ, c->d_jinv, c->d_xsol,
                                                            c->d_krfl, c->phys.kr_scale, c->phys.kr_c[0], c->phys.kr_c[1],
                                                            c->phys.kr_c[2], c->phys.kr_wscale);
  ++c->launches;
  CU(c, cudaGetLastError());
  face_geometry_kernel<<<grid_1d(c, c->E * 6 * c->n2, 256), 256, 0, c->stream>>>(c->n, c->E, c->d_Sfl, c->d_nfc);
  ++c->launches;
  CU(c, cudaGetLastError());
  if (c->d_Sint) {
    interior_S_kernel<<<grid_1d(c, c->E * 9 * c->n2 * (c->n - 1), 256), 256, 0, c->stream>>>(c->n, c->E, c->d_Sfl, c->d_Sint);
    ++c->launches;
    CU(c, cudaGetLastError());
  }
  return CHORUS_OK;
}

template <class T>
int upload(chorus_ctx* c, T** dst, const T* src, size_t count) {
  CU(c, cudaMalloc(dst, sizeof(T) * count));
  CU(c, cudaMemcpyAsync(*dst, src, sizeof(T) * count, cudaMemcpyHostToDevice, c->stream));
  return CHORUS_OK;
}

}  // namespace

extern "C" {

int chorus_init(chorus_ctx** out, const chorus_mesh* mesh, int order, const chorus_physics* phys, void* cuda_stream) {
  if (!out) return CHORUS_EINVAL;
  *out = nullptr;
  if (!mesh || !phys || order < 2 || order > kMaxN || mesh->n_elem <= 0 || mesh->n_geom < 2 || mesh->n_geom > 12 || !mesh->geom_nodes ||
      !mesh->xyz || !mesh->nbr_elem || !mesh->nbr_face || !mesh->nbr_orient)
    return CHORUS_EINVAL;
  for (int64_t i = 0; i < mesh->n_elem * 6; ++i) {
    const int32_t ne = mesh->nbr_elem[i];
    if (ne >= mesh->n_elem || ne < -2 || mesh->nbr_face[i] > 5 || mesh->nbr_orient[i] > 7) return CHORUS_EINVAL;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return CHORUS_ECUDA;   // no device: fail loudly, never fall back
  chorus_ctx* c = new (std::nothrow) chorus_ctx;
  if (!c) return CHORUS_ENOMEM;
  c->n = order; c->n2 = order * order; c->n3 = c->n2 * order; c->nf = c->n2 * (order + 1);
  c->E = mesh->n_elem;
  c->E_own = mesh->n_elem;
  c->ng = mesh->n_geom;
  c->stream = (cudaStream_t)cuda_stream;
  c->phys = *phys;
  c->ph = to_device_phys(*phys);
  auto bail = [&](int rc) {
    chorus_free(c);
    return rc;
  };
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return bail(CHORUS_ECUDA);
  if (const char* kv = std::getenv("CHORUS_KERNELS")) c->use_mma = std::strcmp(kv, "scalar") != 0;
  c->num_sms = prop.multiProcessorCount;
  c->max_smem = prop.sharedMemPerBlockOptin;

  // operator tables: constant memory for the hot kernels, global memory for the geometry kernel
  Basis B = make_basis(order);
  {
    OpsC h;
    std::memset(&h, 0, sizeof h);
    std::memcpy(h.Isf, B.Isf.data(), sizeof(double) * B.Isf.size());
    std::memcpy(h.Dfs, B.Dfs.data(), sizeof(double) * B.Dfs.size());
    std::memcpy(h.Dss, B.Dss.data(), sizeof(double) * B.Dss.size());
    if (cudaMemcpyToSymbolAsync(c_ops, &h, sizeof h, sizeof(OpsC) * order, cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
      return bail(CHORUS_ECUDA);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return bail(CHORUS_ECUDA);   // h is a stack object
  }
  std::vector<double> Gm = geometry_interp(B, mesh->geom_nodes, mesh->n_geom);
  const size_t ng3 = (size_t)c->ng * c->ng * c->ng;
  int rc = 0;
  if ((rc = upload(c, &c->d_Gm, Gm.data(), Gm.size()))) return bail(rc);
  if ((rc = upload(c, &c->d_Dff, B.Dff.data(), B.Dff.size()))) return bail(rc);
  if ((rc = upload(c, &c->d_Efs, B.Efs.data(), B.Efs.size()))) return bail(rc);
  if ((rc = upload(c, &c->d_Dfs, B.Dfs.data(), B.Dfs.size()))) return bail(rc);
  if ((rc = upload(c, &c->d_wq, B.wq.data(), B.wq.size()))) return bail(rc);
  if ((rc = upload(c, &c->d_xyz, mesh->xyz, (size_t)c->E * 3 * ng3))) return bail(rc);
  if ((rc = upload(c, &c->d_nbr_elem, mesh->nbr_elem, (size_t)c->E * 6))) return bail(rc);
  if ((rc = upload(c, &c->d_nbr_face, mesh->nbr_face, (size_t)c->E * 6))) return bail(rc);
  if ((rc = upload(c, &c->d_nbr_orient, mesh->nbr_orient, (size_t)c->E * 6))) return bail(rc);
  const size_t E = (size_t)c->E;
  auto dalloc = [&](double** p, size_t count) { return cudaMalloc(p, sizeof(double) * count) == cudaSuccess; };
  bool ok = dalloc(&c->d_Sfl, E * 9 * c->nf) && dalloc(&c->d_detJ, E * c->n3) && dalloc(&c->d_jinv, E * 9 * c->n3) &&
            dalloc(&c->d_xsol, E * 3 * c->n3) && dalloc(&c->d_nfc, E * 24 * c->n2) && dalloc(&c->d_Qf[0], E * 54 * c->n2) && dalloc(&c->d_Qf[1], E * 54 * c->n2) &&
            dalloc(&c->d_Vf, E * 42 * c->n2);
  if (kSintOrder(c->n)) ok = ok && dalloc(&c->d_Sint, E * 9 * c->n2 * (c->n - 1));
  for (int k = 0; k < 5 && ok; ++k) ok = dalloc(&c->d_U[k], E * 9 * c->n3);
  ok = ok && cudaMalloc(&c->d_ws, sizeof(unsigned long long)) == cudaSuccess;
  ok = ok && dalloc(&c->d_diag, (size_t)(kDiagBlocks + 1) * 3);
  ok = ok && cudaMalloc(&c->d_arrivals, sizeof(unsigned) * 1024) == cudaSuccess &&
       cudaMemsetAsync(c->d_arrivals, 0, sizeof(unsigned) * 1024, c->stream) == cudaSuccess;
  if (!ok) return bail(CHORUS_ENOMEM);
  if ((rc = run_geometry(c))) return bail(rc);
  if (cudaStreamSynchronize(c->stream) != cudaSuccess) return bail(CHORUS_ECUDA);   // host mesh buffers may be released by the caller
  cudaFree(c->d_xyz);   // the geometry nodes are no longer needed unless kappa_r changes; keep a copy only on demand
  c->d_xyz = nullptr;
  *out = c;
  return CHORUS_OK;
}

void chorus_free(chorus_ctx* c) {
  if (!c) return;
  cudaFree(c->d_xyz); cudaFree(c->d_nbr_elem); cudaFree(c->d_nbr_face); cudaFree(c->d_nbr_orient);
  cudaFree(c->d_Gm); cudaFree(c->d_Dff); cudaFree(c->d_Efs); cudaFree(c->d_Dfs);
  cudaFree(c->d_Sfl); cudaFree(c->d_Sint); cudaFree(c->d_detJ); cudaFree(c->d_jinv); cudaFree(c->d_xsol); cudaFree(c->d_krfl); cudaFree(c->d_nfc);
  for (int k = 0; k < 5; ++k) cudaFree(c->d_U[k]);
  cudaFree(c->d_Qf[0]); cudaFree(c->d_Qf[1]); cudaFree(c->d_Vf); cudaFree(c->d_send_elem); cudaFree(c->d_send_face); cudaFree(c->d_recv_elem); cudaFree(c->d_recv_face);
  cudaFree(c->d_ws); cudaFree(c->d_wq); cudaFree(c->d_diag); cudaFree(c->d_arrivals); cudaFree(c->d_scratch);
  for (auto& v : c->prof_ev)
    for (auto& ev : v) {
      cudaEventDestroy(ev.first);
      cudaEventDestroy(ev.second);
    }
  if (HostPipe* hp = c->pipe) {
    if (hp->s_in) cudaStreamSynchronize(hp->s_in);
    if (hp->s_out) cudaStreamSynchronize(hp->s_out);
    for (int k = 0; k < 2; ++k) {
      cudaFree(hp->in[k]); cudaFree(hp->out[k]); cudaFree(hp->ws[k]);
      if (hp->in_ready[k]) cudaEventDestroy(hp->in_ready[k]);
      if (hp->in_free[k]) cudaEventDestroy(hp->in_free[k]);
      if (hp->out_ready[k]) cudaEventDestroy(hp->out_ready[k]);
      if (hp->out_free[k]) cudaEventDestroy(hp->out_free[k]);
    }
    if (hp->s_in) cudaStreamDestroy(hp->s_in);
    if (hp->s_out) cudaStreamDestroy(hp->s_out);
    delete hp;
  }
  delete c;
}

const char* chorus_last_error(const chorus_ctx* c) { return c ? c->err.c_str() : "null context"; }
int64_t chorus_launch_count(const chorus_ctx* c) { return c ? c->launches : 0; }

int chorus_set_physics(chorus_ctx* c, const chorus_physics* phys) {
  if (!c || !phys) return CHORUS_EINVAL;
  if (phys->kr_scale != 0.0 || c->phys.kr_scale != 0.0) {
    const bool same = phys->kr_scale == c->phys.kr_scale && phys->kr_wscale == c->phys.kr_wscale &&
                      std::memcmp(phys->kr_c, c->phys.kr_c, sizeof phys->kr_c) == 0;
    if (!same) return fail(c, CHORUS_EINVAL, "kappa_r parameters are fixed at chorus_init (they are tabulated at the flux points)");
  }
  c->phys = *phys;
  c->ph = to_device_phys(*phys);
  return CHORUS_OK;
}

int chorus_set_state(chorus_ctx* c, const double* q, int on_device) {
  if (!c || !q) return CHORUS_EINVAL;
  const size_t count = (size_t)c->E * 9 * c->n3;
  const double* src = q;
  if (!on_device) {
    CU(c, cudaMemcpyAsync(c->d_U[4], q, sizeof(double) * count, cudaMemcpyHostToDevice, c->stream));
    src = c->d_U[4];
  }
  to_element_major<<<grid_1d(c, (int64_t)count, 256), 256, 0, c->stream>>>(c->E, c->n3, 9, src, c->d_U[0]);
  ++c->launches;
  CU(c, cudaGetLastError());
  if (!on_device) CU(c, cudaStreamSynchronize(c->stream));
  c->cur = 0;
  c->have_state = true;
  c->traces_valid = false;
  return CHORUS_OK;
}

int chorus_get_state(chorus_ctx* c, double* q, int on_device) {
  if (!c || !q) return CHORUS_EINVAL;
  if (!c->have_state) return fail(c, CHORUS_ESTATE, "no state set");
  const size_t count = (size_t)c->E * 9 * c->n3;
  double* dst = on_device ? q : c->d_U[(c->cur + 1) % 5];
  from_element_major<<<grid_1d(c, (int64_t)count, 256), 256, 0, c->stream>>>(c->E, c->n3, 9, c->d_U[c->cur], dst);
  ++c->launches;
  CU(c, cudaGetLastError());
  if (!on_device) {
    CU(c, cudaMemcpyAsync(q, dst, sizeof(double) * count, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
  }
  return CHORUS_OK;
}

int chorus_residual(chorus_ctx* c, double* r, int on_device) {
  if (!c || !r) return CHORUS_EINVAL;
  if (!c->have_state) return fail(c, CHORUS_ESTATE, "no state set");
  if (c->E_own != c->E) return fail(c, CHORUS_EINVAL, "chorus_residual serves whole meshes; a partition advances through the split step");
  if (c->split_next >= 0) return fail(c, CHORUS_ESTATE, "a split step is in progress");
  const size_t count = (size_t)c->E * 9 * c->n3;
  StageOut o{};
  o.Rout = on_device ? r : c->d_U[(c->cur + 1) % 5];
  const double* Qin = c->d_U[c->cur];
  double* scratch = c->d_U[(c->cur + 2) % 5];
  int rc = DISPATCH_N(c, H::stage(c, Qin, o, scratch));
  if (rc) return rc;
  if (!on_device) {
    CU(c, cudaMemcpyAsync(r, o.Rout, sizeof(double) * count, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
  }
  return CHORUS_OK;
}

namespace {
// Stage i (0-based) of an nstages-stage step of size dt on the register ring b[0..4] (b[0] holds the current state):
// which register is evaluated, which receives  sum_k c_k U[A_k] + bdt * R(U[in]),  and which register is current afterwards.
struct StageArgs {
  int in, outb, cur_after;
  const double *A0, *A1, *A2;
  double c0, c1, c2, bdt;
};
bool stage_args(const chorus_ctx* c, int nstages, int i, double dt, const int* b, StageArgs& a) {
  double* const* U = c->d_U;
  a = StageArgs{0, 0, 0, nullptr, nullptr, nullptr, 0.0, 0.0, 0.0, 0.0};
  auto set = [&](int in, int outb, const double* A0, double c0, const double* A1, double c1, const double* A2, double c2, double bdt) {
    a.in = b[in]; a.outb = b[outb]; a.A0 = A0; a.c0 = c0; a.A1 = A1; a.c1 = c1; a.A2 = A2; a.c2 = c2; a.bdt = bdt;
    a.cur_after = b[outb];
  };
  if (nstages == 1) {
    if (i != 0) return false;
    set(0, 1, U[b[0]], 1.0, nullptr, 0, nullptr, 0, dt);
  } else if (nstages == 3) {   // Shu-Osher SSPRK(3,3)
    if (i == 0) set(0, 1, U[b[0]], 1.0, nullptr, 0, nullptr, 0, dt);
    else if (i == 1) set(1, 2, U[b[0]], 0.75, U[b[1]], 0.25, nullptr, 0, 0.25 * dt);
    else if (i == 2) set(2, 3, U[b[0]], 1.0 / 3.0, U[b[2]], 2.0 / 3.0, nullptr, 0, (2.0 / 3.0) * dt);
    else return false;
  } else if (nstages == 5) {
    // SSPRK(5,3) of Ruuth in Shu-Osher form; F(u0) and F(u1) of stages 4 and 5 are eliminated through
    // dt F(u0) = (u1 - u0)/beta1 and dt F(u1) = (u2 - u1)/beta1, so only state registers are kept.
    const double be1 = 0.37726891511710;
    const double a30 = 0.56656131914033, a32 = 0.43343868085967, b32 = 0.16352294089771;
    const double a40 = 0.09299483444413, a41 = 0.00002090369620, a43 = 0.90698426185967, b40 = 0.00071997378654, b43 = 0.34217696850008;
    const double a50 = 0.00736132260920, a51 = 0.20127980325145, a52 = 0.00182955389682, a54 = 0.78952932024253;
    const double b50 = 0.00277719819460, b51 = 0.00001567934613, b54 = 0.29786487010104;
    const double c40 = a40 - b40 / be1, c41 = a41 + b40 / be1;
    const double c50 = a50 - b50 / be1, c51 = a51 + b50 / be1 - b51 / be1, c52 = a52 + b51 / be1;
    (void)c50;   // = -4e-16: u0's weight in stage 5 cancels to round-off and is dropped
    if (i == 0) set(0, 1, U[b[0]], 1.0, nullptr, 0, nullptr, 0, be1 * dt);
    else if (i == 1) set(1, 2, U[b[1]], 1.0, nullptr, 0, nullptr, 0, be1 * dt);
    else if (i == 2) set(2, 3, U[b[0]], a30, U[b[2]], a32, nullptr, 0, b32 * dt);
    else if (i == 3) set(3, 4, U[b[0]], c40, U[b[1]], c41, U[b[3]], a43, b43 * dt);
    else if (i == 4) set(4, 0, U[b[1]], c51, U[b[2]], c52, U[b[4]], a54, b54 * dt);
    else return false;
  } else {
    return false;
  }
  return true;
}
int run_stage(chorus_ctx* c, const StageArgs& a, bool split) {
  StageOut o{};
  o.Qout = c->d_U[a.outb];
  o.A0 = a.A0; o.A1 = a.A1; o.A2 = a.A2;
  o.c0 = a.c0; o.c1 = a.c1; o.c2 = a.c2; o.bdt = a.bdt;
  const double* Qin = c->d_U[a.in];
  return DISPATCH_N(c, H::stage(c, Qin, o, nullptr, split));
}
}  // namespace

int chorus_step(chorus_ctx* c, double dt, int nstages) {
  if (!c || (nstages != 1 && nstages != 3 && nstages != 5) || !(dt == dt)) return c ? fail(c, CHORUS_EINVAL, "bad dt or nstages") : CHORUS_EINVAL;
  if (!c->have_state) return fail(c, CHORUS_ESTATE, "no state set");
  if (c->E_own != c->E) return fail(c, CHORUS_EINVAL, "a partition steps through chorus_step_begin / chorus_stage_main / chorus_stage_face");
  if (c->split_next >= 0) return fail(c, CHORUS_ESTATE, "a split step is in progress");
  int b[5];
  for (int k = 0; k < 5; ++k) b[k] = (c->cur + k) % 5;
  // a stage that fails leaves the trace buffers describing an intermediate state: they must not be reused
  struct TraceGuard {
    chorus_ctx* c;
    bool ok = false;
    ~TraceGuard() { if (!ok) c->traces_valid = false; }
  } guard{c};
  StageArgs a;
  for (int i = 0; i < nstages; ++i) {
    stage_args(c, nstages, i, dt, b, a);
    int rc = run_stage(c, a, false);
    if (rc) return rc;
  }
  c->cur = a.cur_after;
  guard.ok = true;
  return CHORUS_OK;
}

// ---- host jobs, pipelined: H2D of job k + 1 and D2H of job k - 1 run beside the kernels of job k
namespace {
int host_pipe(chorus_ctx* c, HostPipe** out) {
  if (!c->pipe) {
    HostPipe* hp = new HostPipe;
    c->pipe = hp;                    // chorus_free releases whatever was made, also after a failure below
    const size_t count = (size_t)c->E * 9 * c->n3;
    CU(c, cudaStreamCreateWithFlags(&hp->s_in, cudaStreamNonBlocking));
    CU(c, cudaStreamCreateWithFlags(&hp->s_out, cudaStreamNonBlocking));
    for (int k = 0; k < 2; ++k) {
      if (cudaMalloc(&hp->in[k], sizeof(double) * count) != cudaSuccess || cudaMalloc(&hp->out[k], sizeof(double) * count) != cudaSuccess ||
          cudaMalloc(&hp->ws[k], sizeof(unsigned long long)) != cudaSuccess)
        return fail(c, CHORUS_ENOMEM, "chorus_step_host: staging buffers");
      CU(c, cudaEventCreateWithFlags(&hp->in_ready[k], cudaEventDisableTiming));
      CU(c, cudaEventCreateWithFlags(&hp->in_free[k], cudaEventDisableTiming));
      CU(c, cudaEventCreateWithFlags(&hp->out_ready[k], cudaEventDisableTiming));
      CU(c, cudaEventCreateWithFlags(&hp->out_free[k], cudaEventDisableTiming));
    }
  }
  if (!c->pipe->out_free[1]) return fail(c, CHORUS_ESTATE, "chorus_step_host: the pipeline could not be set up earlier");
  *out = c->pipe;
  return CHORUS_OK;
}
}  // namespace

int chorus_step_host(chorus_ctx* c, const double* q_in, double* q_out, double dt, int nstages, double* ws_out) {
  if (!c || !q_in || !q_out) return CHORUS_EINVAL;
  if ((nstages != 1 && nstages != 3 && nstages != 5) || !(dt == dt)) return fail(c, CHORUS_EINVAL, "bad dt or nstages");
  if (c->E_own != c->E) return fail(c, CHORUS_EINVAL, "chorus_step_host serves unpartitioned contexts");
  if (c->split_next >= 0) return fail(c, CHORUS_ESTATE, "a split step is in progress");
  HostPipe* hp = nullptr;
  if (int rc = host_pipe(c, &hp)) return rc;
  const int k = (int)(hp->jobs & 1);
  const bool reuse = hp->jobs >= 2;                       // slot k was last used by job jobs - 2
  const size_t count = (size_t)c->E * 9 * c->n3;
  // copy-in stream: the staged input of slot k must have been consumed (transposed into the state registers) by its last job
  if (reuse) CU(c, cudaStreamWaitEvent(hp->s_in, hp->in_free[k], 0));
  CU(c, cudaMemcpyAsync(hp->in[k], q_in, sizeof(double) * count, cudaMemcpyHostToDevice, hp->s_in));
  CU(c, cudaEventRecord(hp->in_ready[k], hp->s_in));
  // the context's stream: state in, one step, state (and wave speed) out
  CU(c, cudaStreamWaitEvent(c->stream, hp->in_ready[k], 0));
  to_element_major<<<grid_1d(c, (int64_t)count, 256), 256, 0, c->stream>>>(c->E, c->n3, 9, hp->in[k], c->d_U[0]);
  ++c->launches;
  CU(c, cudaGetLastError());
  CU(c, cudaEventRecord(hp->in_free[k], c->stream));
  c->cur = 0;
  c->have_state = true;
  c->traces_valid = false;
  if (int rc = chorus_step(c, dt, nstages)) return rc;
  if (reuse) CU(c, cudaStreamWaitEvent(c->stream, hp->out_free[k], 0));      // the D2H of slot k's last result has finished
  from_element_major<<<grid_1d(c, (int64_t)count, 256), 256, 0, c->stream>>>(c->E, c->n3, 9, c->d_U[c->cur], hp->out[k]);
  ++c->launches;
  CU(c, cudaGetLastError());
  if (ws_out) {
    CU(c, cudaMemsetAsync(hp->ws[k], 0, sizeof(unsigned long long), c->stream));
    const int64_t total = c->E * c->n3;
    wavespeed_kernel<<<grid_1d(c, total, 256), 256, 0, c->stream>>>(c->E, c->n3, c->ph, c->d_U[c->cur], hp->ws[k]);
    ++c->launches;
    CU(c, cudaGetLastError());
  }
  CU(c, cudaEventRecord(hp->out_ready[k], c->stream));
  // copy-out stream
  CU(c, cudaStreamWaitEvent(hp->s_out, hp->out_ready[k], 0));
  CU(c, cudaMemcpyAsync(q_out, hp->out[k], sizeof(double) * count, cudaMemcpyDeviceToHost, hp->s_out));
  if (ws_out) CU(c, cudaMemcpyAsync(ws_out, hp->ws[k], sizeof(double), cudaMemcpyDeviceToHost, hp->s_out));
  CU(c, cudaEventRecord(hp->out_free[k], hp->s_out));
  ++hp->jobs;
  return CHORUS_OK;
}

int chorus_sync(chorus_ctx* c) {
  if (!c) return CHORUS_EINVAL;
  if (c->pipe && c->pipe->s_in) CU(c, cudaStreamSynchronize(c->pipe->s_in));
  CU(c, cudaStreamSynchronize(c->stream));
  if (c->pipe && c->pipe->s_out) CU(c, cudaStreamSynchronize(c->pipe->s_out));
  return CHORUS_OK;
}

// ---- the same step, one kernel at a time (what a partition's driver interleaves with its halo exchanges)
int chorus_step_begin(chorus_ctx* c, double dt, int nstages) {
  if (!c || (nstages != 1 && nstages != 3 && nstages != 5) || !(dt == dt)) return c ? fail(c, CHORUS_EINVAL, "bad dt or nstages") : CHORUS_EINVAL;
  if (!c->have_state) return fail(c, CHORUS_ESTATE, "no state set");
  if (c->split_next >= 0) return fail(c, CHORUS_ESTATE, "a split step is already in progress");
  const double* Qin = c->d_U[c->cur];
  int rc = DISPATCH_N(c, H::ensure_traces(c, Qin));
  if (rc) return rc;
  for (int k = 0; k < 5; ++k) c->split_b[k] = (c->cur + k) % 5;
  c->split_dt = dt;
  c->split_nstages = nstages;
  c->split_next = 0;
  c->split_face_pending = false;
  return CHORUS_OK;
}

int chorus_stage_main(chorus_ctx* c, int istage) {
  if (!c) return CHORUS_EINVAL;
  if (c->split_next < 0 || istage != c->split_next || c->split_face_pending) return fail(c, CHORUS_ESTATE, "chorus_stage_main out of sequence");
  StageArgs a;
  if (!stage_args(c, c->split_nstages, istage, c->split_dt, c->split_b, a)) return fail(c, CHORUS_EINVAL, "bad stage index");
  int rc = run_stage(c, a, true);
  if (rc) {
    c->traces_valid = false;
    c->split_next = -1;
    return rc;
  }
  c->split_face_pending = true;
  return CHORUS_OK;
}

int chorus_stage_face(chorus_ctx* c, int istage) {
  if (!c) return CHORUS_EINVAL;
  if (c->split_next < 0 || istage != c->split_next || !c->split_face_pending) return fail(c, CHORUS_ESTATE, "chorus_stage_face out of sequence");
  int rc = DISPATCH_N(c, H::face_pending(c));
  c->split_face_pending = false;
  if (rc) {
    c->traces_valid = false;
    c->split_next = -1;
    return rc;
  }
  if (istage + 1 == c->split_nstages) {
    StageArgs a;
    stage_args(c, c->split_nstages, istage, c->split_dt, c->split_b, a);
    c->cur = a.cur_after;
    c->split_next = -1;
  } else {
    c->split_next = istage + 1;
  }
  return CHORUS_OK;
}

// ---- partitions: owned elements first, ghosts after; halo faces packed into / unpacked from contiguous device buffers
int chorus_set_owned(chorus_ctx* c, int64_t n_owned) {
  if (!c || n_owned < 1 || n_owned > c->E) return c ? fail(c, CHORUS_EINVAL, "n_owned must be in 1..n_elem") : CHORUS_EINVAL;
  c->E_own = n_owned;
  c->traces_valid = false;
  return CHORUS_OK;
}

int chorus_halo_setup(chorus_ctx* c, int64_t n_send, const int32_t* send_elem, const uint8_t* send_face, int64_t n_recv,
                      const int32_t* recv_elem, const uint8_t* recv_face) {
  if (!c || n_send < 0 || n_recv < 0 || (n_send && (!send_elem || !send_face)) || (n_recv && (!recv_elem || !recv_face))) return CHORUS_EINVAL;
  for (int64_t k = 0; k < n_send; ++k)
    if (send_elem[k] < 0 || send_elem[k] >= c->E_own || send_face[k] > 5) return fail(c, CHORUS_EINVAL, "halo send list: owned element and face 0..5");
  for (int64_t k = 0; k < n_recv; ++k)
    if (recv_elem[k] < c->E_own || recv_elem[k] >= c->E || recv_face[k] > 5) return fail(c, CHORUS_EINVAL, "halo receive list: ghost element and face 0..5");
  cudaFree(c->d_send_elem); cudaFree(c->d_send_face); cudaFree(c->d_recv_elem); cudaFree(c->d_recv_face);
  c->d_send_elem = c->d_recv_elem = nullptr;
  c->d_send_face = c->d_recv_face = nullptr;
  c->n_send = c->n_recv = 0;
  int rc = 0;
  if (n_send && ((rc = upload(c, &c->d_send_elem, send_elem, (size_t)n_send)) || (rc = upload(c, &c->d_send_face, send_face, (size_t)n_send)))) return rc;
  if (n_recv && ((rc = upload(c, &c->d_recv_elem, recv_elem, (size_t)n_recv)) || (rc = upload(c, &c->d_recv_face, recv_face, (size_t)n_recv)))) return rc;
  CU(c, cudaStreamSynchronize(c->stream));   // the host lists may be released by the caller
  c->n_send = n_send;
  c->n_recv = n_recv;
  return CHORUS_OK;
}

namespace {
// field 0: face traces of the current state (9 n^2 doubles per face); field 1: own-side viscous face fluxes (7 n^2)
int halo_copy(chorus_ctx* c, int field, double* buf, bool pack) {
  if (!c || (field != 0 && field != 1) || !buf) return c ? fail(c, CHORUS_EINVAL, "halo field 0 (traces) or 1 (viscous face fluxes)") : CHORUS_EINVAL;
  const int64_t cnt = pack ? c->n_send : c->n_recv;
  if (cnt == 0) return CHORUS_OK;
  const int w = (field == 0 ? 9 : 7) * c->n2;
  double* base = field == 0 ? c->d_Qf[c->qf_cur] : c->d_Vf;
  const int32_t* el = pack ? c->d_send_elem : c->d_recv_elem;
  const uint8_t* fc = pack ? c->d_send_face : c->d_recv_face;
  halo_copy_kernel<<<grid_1d(c, cnt * w, 256), 256, 0, c->stream>>>(cnt, w, el, fc, base, buf, pack ? 1 : 0);
  ++c->launches;
  CU(c, cudaGetLastError());
  return CHORUS_OK;
}
}  // namespace

int chorus_halo_pack(chorus_ctx* c, int field, double* buf) { return halo_copy(c, field, buf, true); }
int chorus_halo_unpack(chorus_ctx* c, int field, const double* buf) { return halo_copy(c, field, const_cast<double*>(buf), false); }

int chorus_max_wavespeed(chorus_ctx* c, double* out) {
  if (!c || !out) return CHORUS_EINVAL;
  if (!c->have_state) return fail(c, CHORUS_ESTATE, "no state set");
  CU(c, cudaMemsetAsync(c->d_ws, 0, sizeof(unsigned long long), c->stream));
  const int64_t total = c->E_own * c->n3;
  int grid = grid_1d(c, total, 256);
  wavespeed_kernel<<<grid, 256, 0, c->stream>>>(c->E_own, c->n3, c->ph, c->d_U[c->cur], c->d_ws);
  ++c->launches;
  CU(c, cudaGetLastError());
  unsigned long long bits = 0;
  CU(c, cudaMemcpyAsync(&bits, c->d_ws, sizeof bits, cudaMemcpyDeviceToHost, c->stream));
  CU(c, cudaStreamSynchronize(c->stream));
  double v;
  std::memcpy(&v, &bits, sizeof v);
  *out = v;
  if (!std::isfinite(v)) return fail(c, CHORUS_ESTATE, "non-finite wave speed");
  return CHORUS_OK;
}

namespace {
int diagnostics_impl(chorus_ctx* c, double* out, bool sums) {
  if (!c || !out) return CHORUS_EINVAL;
  if (!c->have_state) return fail(c, CHORUS_ESTATE, "no state set");
  const int64_t total = c->E_own * c->n3;
  const int grid = (int)std::min<int64_t>(kDiagBlocks, (total + 255) / 256);
  diagnostics_kernel<<<grid, 256, 0, c->stream>>>(c->E_own, c->n, c->d_wq, c->d_detJ, c->d_U[c->cur], c->d_diag);
  ++c->launches;
  CU(c, cudaGetLastError());
  diagnostics_final_kernel<<<1, 256, 0, c->stream>>>(grid, c->d_diag, c->d_diag + (size_t)kDiagBlocks * 3, sums ? 1 : 0);
  ++c->launches;
  CU(c, cudaGetLastError());
  CU(c, cudaMemcpyAsync(out, c->d_diag + (size_t)kDiagBlocks * 3, sizeof(double) * 3, cudaMemcpyDeviceToHost, c->stream));
  CU(c, cudaStreamSynchronize(c->stream));
  return CHORUS_OK;
}
}  // namespace
int chorus_diagnostics(chorus_ctx* c, double* out) { return diagnostics_impl(c, out, false); }
int chorus_diagnostics_sums(chorus_ctx* c, double* out) { return diagnostics_impl(c, out, true); }

int chorus_get_geometry(chorus_ctx* c, double* detJ, double* S, double* xsol, double* jinv, int on_device) {
  if (!c) return CHORUS_EINVAL;
  const size_t E = (size_t)c->E;
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  if (detJ) CU(c, cudaMemcpyAsync(detJ, c->d_detJ, sizeof(double) * E * c->n3, kind, c->stream));
  if (S) CU(c, cudaMemcpyAsync(S, c->d_Sfl, sizeof(double) * E * 9 * c->nf, kind, c->stream));
  if (jinv) CU(c, cudaMemcpyAsync(jinv, c->d_jinv, sizeof(double) * E * 9 * c->n3, kind, c->stream));
  if (xsol) {
    const size_t count = E * 3 * c->n3;
    double* dst = on_device ? xsol : c->d_U[(c->cur + 1) % 5];
    from_element_major<<<grid_1d(c, (int64_t)count, 256), 256, 0, c->stream>>>(c->E, c->n3, 3, c->d_xsol, dst);
    ++c->launches;
    CU(c, cudaGetLastError());
    if (!on_device) CU(c, cudaMemcpyAsync(xsol, dst, sizeof(double) * count, cudaMemcpyDeviceToHost, c->stream));
  }
  if (!on_device) CU(c, cudaStreamSynchronize(c->stream));
  return CHORUS_OK;
}

int chorus_get_gradient(chorus_ctx* c, double* g, int on_device) {
  if (!c || !g) return CHORUS_EINVAL;
  if (!c->have_state) return fail(c, CHORUS_ESTATE, "no state set");
  const size_t count = (size_t)c->E * 27 * c->n3;
  double *tmp = nullptr, *tmp2 = nullptr;
  CU(c, cudaMalloc(&tmp, sizeof(double) * count));
  if (!on_device && cudaMalloc(&tmp2, sizeof(double) * count) != cudaSuccess) {
    cudaFree(tmp);
    return fail(c, CHORUS_ENOMEM, "gradient scratch");
  }
  const double* Qin = c->d_U[c->cur];
  c->traces_valid = false;   // d_Qf[0] is used as scratch below
  c->qf_cur = 0;
  int rc = DISPATCH_N(c, H::trace(c, Qin, c->d_Qf[0]));
  if (!rc) rc = DISPATCH_N(c, H::grad(c, Qin, nullptr, tmp));
  if (!rc) {
    double* dst = on_device ? g : tmp2;
    from_element_major<<<grid_1d(c, (int64_t)count, 256), 256, 0, c->stream>>>(c->E, c->n3, 27, tmp, dst);
    ++c->launches;
    if (cudaGetLastError() != cudaSuccess) rc = fail(c, CHORUS_ECUDA, "from_element_major launch");
    if (!rc && !on_device && cudaMemcpyAsync(g, dst, sizeof(double) * count, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
      rc = fail(c, CHORUS_ECUDA, "gradient copy");
  }
  if (cudaStreamSynchronize(c->stream) != cudaSuccess && !rc) rc = fail(c, CHORUS_ECUDA, "stream sync");
  cudaFree(tmp);
  cudaFree(tmp2);
  return rc;
}

int chorus_profile(chorus_ctx* c, int enable) {
  if (!c) return CHORUS_EINVAL;
  c->prof = enable != 0;
  return CHORUS_OK;
}

int chorus_profile_read(chorus_ctx* c, double* ms, int64_t* launches) {
  if (!c || !ms || !launches) return CHORUS_EINVAL;
  CU(c, cudaStreamSynchronize(c->stream));
  for (int k = 0; k < 3; ++k) {
    double tot = 0.0;
    for (auto& ev : c->prof_ev[k]) {
      float t = 0.f;
      cudaEventElapsedTime(&t, ev.first, ev.second);
      tot += t;
      cudaEventDestroy(ev.first);
      cudaEventDestroy(ev.second);
    }
    ms[k] = tot;
    launches[k] = (int64_t)c->prof_ev[k].size();
    c->prof_ev[k].clear();
  }
  return CHORUS_OK;
}

int chorus_fp64_peak(int mode, double seconds, double* tflops, double* dfma_tflops, double* dmma_tflops) {
  if (mode < 0 || mode > 2 || !tflops || !(seconds > 0.0)) return CHORUS_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return CHORUS_ECUDA;
  double* out = nullptr;
  if (cudaMalloc(&out, sizeof(double)) != cudaSuccess) return CHORUS_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int grid = sms * 8, iters = 4096;
  auto launch = [&]() {
    if (mode == 0) fp64_peak_kernel<0><<<grid, 256>>>(iters, 1.0, out);
    else if (mode == 1) fp64_peak_kernel<1><<<grid, 256>>>(iters, 1.0, out);
    else fp64_peak_kernel<2><<<grid, 256>>>(iters, 1.0, out);
  };
  launch();   // warm-up
  cudaDeviceSynchronize();
  // flops of one launch: DFMA warps 64 FMA/thread/iter; DMMA warps 8 x 256 FMA/warp/iter = 64 FMA/thread/iter as well
  const double flop_per_launch = 2.0 * 64.0 * 256.0 * (double)grid * iters;
  int reps = 1;
  float ms = 0.f;
  for (;;) {
    cudaEventRecord(e0);
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms * 1e-3 >= seconds || reps > (1 << 20)) break;
    reps *= 2;
  }
  const cudaError_t err = cudaGetLastError();
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (err != cudaSuccess || ms <= 0.f) return CHORUS_ECUDA;
  *tflops = flop_per_launch * reps / (ms * 1e-3) / 1e12;
  if (dfma_tflops) *dfma_tflops = mode == 0 ? *tflops : mode == 2 ? 0.5 * *tflops : 0.0;
  if (dmma_tflops) *dmma_tflops = mode == 1 ? *tflops : mode == 2 ? 0.5 * *tflops : 0.0;
  return CHORUS_OK;
}

int chorus_get_operators(int order, double* xs, double* xf, double* Isf, double* Dfs) {
  if (order < 2 || order > kMaxN) return CHORUS_EINVAL;
  Basis B = make_basis(order);
  if (xs) std::memcpy(xs, B.xs.data(), sizeof(double) * B.xs.size());
  if (xf) std::memcpy(xf, B.xf.data(), sizeof(double) * B.xf.size());
  if (Isf) std::memcpy(Isf, B.Isf.data(), sizeof(double) * B.Isf.size());
  if (Dfs) std::memcpy(Dfs, B.Dfs.data(), sizeof(double) * B.Dfs.size());
  return CHORUS_OK;
}

}  // extern "C"

// =========================================================================================================
// Allocation-free diagnostics (chorus_diagnostics_static, include/chorus.h): for callers that cannot call cudaMalloc (code
// under CUDA graph capture, tight serving loops, harnesses that forbid it).  The partial sums of the reduction -- the scratch
// that chorus_diagnostics keeps in a cudaMalloc'ed buffer of its context -- live in a file-scope device array of fixed size,
// which every GPU that loads the library holds until exit (96 KB).  No context, no cudaMalloc / cudaFree, no host heap use.
//
// The array's NAME is, in host code, a host-side stand-in and not a device address: the address the kernels are given is
// obtained once per device, with that device current, by cudaGetSymbolAddress (static_diag_scratch below).
// =========================================================================================================
namespace {
constexpr int kStaticDiagPointsPerBlock = 8192;      // solution points summed by one block (fixed: the summation tree depends on the size only)
constexpr int kStaticDiagMaxBlocks = CHORUS_STATIC_DIAG_MAX_POINTS / kStaticDiagPointsPerBlock;   // 4096 partial triples
static_assert((int64_t)kStaticDiagMaxBlocks * kStaticDiagPointsPerBlock == CHORUS_STATIC_DIAG_MAX_POINTS, "maximum = whole blocks");
}  // namespace

// partial sums [block][3] of one call.  Shared by every call on the device; keeps the last call's contents.
static __device__ __align__(256) double g_static_diag_scratch[kStaticDiagMaxBlocks * 3];

namespace chorus {
struct QuadW { double w[kMaxN]; };   // quadrature weights of the solution points, by value (no device copy to allocate)

// Variant of diagnostics_kernel: the state in the INTERFACE layout [9][E][n3] (what the caller holds), weights by value, a fixed
// chunk of points per block, partial sums into the static scratch.  Every partial the final kernel reads is written by this
// launch: nothing in the scratch has to start at zero.
__global__ void __launch_bounds__(256) diagnostics_static_kernel(int64_t total, int64_t E, int n, QuadW wq, const double* __restrict__ detJ,
                                                                const double* __restrict__ Q, double* __restrict__ partial) {
  __shared__ double sh[8][3];
  const int n3 = n * n * n;
  const int64_t comp = E * n3;                      // stride between conserved variables
  double V = 0.0, KE = 0.0, EB = 0.0;
  const int64_t t0 = (int64_t)blockIdx.x * kStaticDiagPointsPerBlock;
  const int64_t t1 = t0 + kStaticDiagPointsPerBlock < total ? t0 + kStaticDiagPointsPerBlock : total;
  for (int64_t t = t0 + threadIdx.x; t < t1; t += blockDim.x) {
    const int s = (int)(t % n3);
    const int i = s % n, j = (s / n) % n, k = s / (n * n);
    const double wJ = wq.w[i] * wq.w[j] * wq.w[k] * detJ[t];
    const double* q = Q + t;
    const double rho = q[0], m1 = q[comp], m2 = q[2 * comp], m3 = q[3 * comp];
    const double b1 = q[5 * comp], b2 = q[6 * comp], b3 = q[7 * comp];
    V += wJ;
    KE += wJ * (0.5 * (m1 * m1 + m2 * m2 + m3 * m3) / rho);       // Eq. 34
    EB += wJ * (0.5 * (b1 * b1 + b2 * b2 + b3 * b3));             // Eq. 35
  }
  block_sum3(V, KE, EB, sh);
  if (threadIdx.x == 0) { partial[blockIdx.x * 3 + 0] = V; partial[blockIdx.x * 3 + 1] = KE; partial[blockIdx.x * 3 + 2] = EB; }
}
}  // namespace chorus

namespace {
constexpr int kStaticMaxDevices = 64;
double* g_static_diag_ptr[kStaticMaxDevices] = {};   // device address of g_static_diag_scratch, per device (set-up once)
bool g_static_diag_have[kStaticMaxDevices] = {};
thread_local char g_static_err[256] = "";            // message of the calling thread's last failed context-free call

int static_fail(int code, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) std::snprintf(g_static_err, sizeof g_static_err, "%s: %s", what, cudaGetErrorString(e));
  else std::snprintf(g_static_err, sizeof g_static_err, "%s", what);
  return code;
}

// Set-up, once per device, with that device current: the device address of the scratch array.
int static_diag_scratch(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return static_fail(CHORUS_ECUDA, "cudaGetDevice", e);
  if (dev < 0 || dev >= kStaticMaxDevices) return static_fail(CHORUS_EINVAL, "chorus_diagnostics_static: device ordinal beyond 63");
  if (!__atomic_load_n(&g_static_diag_have[dev], __ATOMIC_ACQUIRE)) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_diag_scratch);
    if (e != cudaSuccess || !p) return static_fail(CHORUS_ECUDA, "cudaGetSymbolAddress(static diagnostics scratch)", e);
    g_static_diag_ptr[dev] = p;      // two threads racing here store the same address
    __atomic_store_n(&g_static_diag_have[dev], true, __ATOMIC_RELEASE);
  }
  *out = g_static_diag_ptr[dev];
  return CHORUS_OK;
}
}  // namespace

extern "C" {

int chorus_diagnostics_static(int order, int64_t n_elem, const double* q, const double* detJ, double* out, void* cuda_stream) {
  g_static_err[0] = '\0';
  if (order < 2 || order > kMaxN) return static_fail(CHORUS_EINVAL, "chorus_diagnostics_static: order must be 2..9");
  if (n_elem <= 0) return static_fail(CHORUS_EINVAL, "chorus_diagnostics_static: n_elem must be positive");
  if (!q || !detJ || !out) return static_fail(CHORUS_EINVAL, "chorus_diagnostics_static: null pointer");
  const int n = order, n3 = n * n * n;
  if (n_elem > CHORUS_STATIC_DIAG_MAX_POINTS / n3) {
    std::snprintf(g_static_err, sizeof g_static_err,
                  "chorus_diagnostics_static: %lld elements x %d points exceed the static scratch's maximum of %d solution points "
                  "(use chorus_diagnostics of a context for larger meshes)", (long long)n_elem, n3, (int)CHORUS_STATIC_DIAG_MAX_POINTS);
    return CHORUS_EINVAL;
  }
  double* scratch = nullptr;
  if (int rc = static_diag_scratch(&scratch)) return rc;
  // Fejer's first rule on the Chebyshev-Gauss points (the closed form of basis.h), on the stack
  QuadW wq;
  const long double pi = 3.14159265358979323846264338327950288L;
  for (int k = 1; k <= kMaxN; ++k) {
    long double w = 0;
    if (k <= n) {
      const long double th = (2 * k - 1) * pi / (2 * n);
      w = 1;
      for (int j = 1; j <= n / 2; ++j) w -= 2 * cosl(2 * j * th) / (4.0L * j * j - 1);
      w /= n;
    }
    wq.w[k - 1] = (double)w;
  }
  const int64_t total = n_elem * n3;
  const int grid = (int)((total + kStaticDiagPointsPerBlock - 1) / kStaticDiagPointsPerBlock);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  diagnostics_static_kernel<<<grid, 256, 0, st>>>(total, n_elem, n, wq, detJ, q, scratch);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return static_fail(CHORUS_ECUDA, "diagnostics_static_kernel launch", e);
  diagnostics_final_kernel<<<1, 256, 0, st>>>(grid, scratch, out, 0);
  e = cudaGetLastError();
  if (e != cudaSuccess) return static_fail(CHORUS_ECUDA, "diagnostics_final_kernel launch", e);
  return CHORUS_OK;
}

const char* chorus_static_last_error(void) { return g_static_err; }

}  // extern "C"
