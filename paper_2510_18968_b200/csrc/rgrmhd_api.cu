// rgrmhd_api.cu -- host driver and C-ABI (include/rgrmhd.h) of the B200-native resistive GRMHD step.
// Stage sequencing of IMEX-SSP2(2,2,2) (Eq. 35-37), device buffers, stream.
// There is no CPU fallback: every step of the path runs in the kernels of this library.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <functional>
#include <vector>

#include "../../include/rgrmhd.h"
#include "rgrmhd_common.cuh"

namespace rg {
cudaError_t launch_c2p(const GridView& G, int stage, double dt, StatsDev* stats, cudaStream_t st);
cudaError_t launch_prim2cons(const GridView& G, cudaStream_t st);
cudaError_t launch_metric_coeffs(const GridView& G, bool store, cudaStream_t st);
cudaError_t launch_rhs_simple(const GridView& G, double dt, int stage, int recon, cudaStream_t st);
cudaError_t launch_rhs_pencil(const GridView& G, double dt, int stage, int recon, int sm_count, cudaStream_t st);
bool rhs_pencil_supported(const GridView& G);
cudaError_t launch_rhs_tma(const GridView& G, const void* state, double dt, int stage, int recon, int sm_count, cudaStream_t st);
void* tma_create(const GridView& G);
void tma_destroy(void* state);
cudaError_t launch_ghost_fill(const GridView& G, double* const* fields, int nf, cudaStream_t st);
cudaError_t launch_halo_copy(const GridView& G, double* const* fields, int nf, int dir, int side, double* buf, bool pack,
                             cudaStream_t st);
cudaError_t launch_charge_div_e(const GridView& G, int stage, double dt, cudaStream_t st);
cudaError_t launch_max_speed(const GridView& G, unsigned long long* out, bool have_prims, int sm_count, cudaStream_t st);
}  // namespace rg

namespace rg {
struct AccTab { double* f[NCONS]; };
struct StageGen {           // mirrors rgrmhd_imex_gen.cu
  int stage, nstages, use_dprev, init;
  double aii, w_dprev[5], w_src[5], w_stiff[5];
  AccTab acc[5];
};
cudaError_t launch_stage_gen(const GridView& G, const StageGen& W, double dt, StatsDev* stats, cudaStream_t st);
cudaError_t launch_charge_sources_gen(const GridView& G, const StageGen& W, double dt, cudaStream_t st);
}  // namespace rg

struct rgrmhd_s {
  rgrmhd_params par;
  rg::GridView G;
  int device = 0;
  cudaStream_t stream = nullptr;
  double* slab = nullptr;            // all fields, one allocation
  double* slab_src = nullptr;        // the static source-coefficient fields that are not identically zero (set_metric)
  int nsrc_fields = 0;
  double* slab2 = nullptr;           // accumulators of the 3rd / 4th stage of the general tableau driver (allocated on first use)
  long long field_stride = 0;        // doubles between consecutive fields (ntot rounded up to 32)
  rg::StatsDev* stats_dev = nullptr;
  unsigned long long* maxspeed_dev = nullptr;
  long long solves = 0;              // host-side count of cell solves enqueued
  long long launches = 0;
  bool have_metric = false, have_prims = false, have_sigma = false;
  bool pending_final = false;   // the last step's final recovery (k_c2p<3>) has not been launched yet
  bool poisoned = false;        // a launch inside rgrmhd_step failed: the state is half advanced until set_prims replaces it
  int sm_count = 148;           // multiprocessors of the device (grid sizing of the flux and reduction kernels)
  bool charge_final_due = false;   // charge mode DIV_E: q, calQ of the new state not computed yet (done on output)
  int part = 0;                      // split step in flight: the part rgrmhd_step_continue runs next (0: none)
  double cur_dt = 0.0; int cur_recon = 0;
  bool maxspeed_fused = false;       // wave mode MHD_INSIDE: the word holds the reduction over the CURRENT state (final recovery)
  bool maxspeed_cached = false;      // wave mode LIGHT: the reduction depends on the metric only (Eq. 30): reuse it
  double maxspeed_value = 0.0;
  int last_rhs_variant = -1;    // flux kernel the last rgrmhd_step actually launched
  int rhs_variant = 0;               // 0 = TMA-staged (default), 1 = simple, 2 = pencil (global-memory stencils)
  void* tma = nullptr;               // tensor maps of the TMA-staged flux kernel (null: shape not supported)
  bool timing = false;
  struct Timed { int cls; cudaEvent_t a, b; };
  std::vector<Timed> timed;
  std::string last_error;
};

namespace {

struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; }
    if (prev != dev) ok = (cudaSetDevice(dev) == cudaSuccess);
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int fail_cuda(rgrmhd_t h, cudaError_t e, const char* what) {
  if (h) h->last_error = std::string(what) + ": " + cudaGetErrorString(e);
  return RGRMHD_E_CUDA;
}

#define RG_CUDA(h, call)                                            \
  do {                                                              \
    cudaError_t e__ = (call);                                       \
    if (e__ != cudaSuccess) return fail_cuda((h), e__, #call);      \
  } while (0)

}  // namespace

extern "C" {

int rgrmhd_params_default(rgrmhd_params* p) {
  if (!p) return RGRMHD_E_INVALID;
  std::memset(p, 0, sizeof(*p));
  for (int d = 0; d < 3; ++d) { p->n[d] = 1; p->dx[d] = 1.0; p->bc[d] = RGRMHD_BC_OUTFLOW; }
  p->ng = 3;
  p->gamma_eos = 4.0 / 3.0;
  p->sigma_model = RGRMHD_SIGMA_UNIFORM;
  p->sigma0 = 0.0; p->sigma_exp = 0.0; p->sigma_dref = 1.0;
  p->kappa = 1.0;
  p->rho_floor = 0.0; p->k_atmo = 0.0;
  p->c2p_tol = 0.0; p->c2p_max_iter = 0;
  p->charge_mode = RGRMHD_CHARGE_CELL_CURRENT;
  p->weno_eps = 0.0;
  p->device = 0;
  return RGRMHD_OK;
}

int rgrmhd_create(rgrmhd_t* out, const rgrmhd_params* p) {
  if (!out || !p) return RGRMHD_E_INVALID;
  *out = nullptr;
  if (p->ng != 3 || !(p->gamma_eos > 1.0)) return RGRMHD_E_INVALID;
  for (int d = 0; d < 3; ++d) {
    if (p->n[d] < 1) return RGRMHD_E_INVALID;
    if (p->n[d] > 1 && !(p->dx[d] > 0.0)) return RGRMHD_E_INVALID;
    if (p->n[d] > 1 && p->n[d] < 3) return RGRMHD_E_INVALID;   // periodic wrap of 3 ghosts needs >= 3 cells
    if (p->bc[d] != RGRMHD_BC_PERIODIC && p->bc[d] != RGRMHD_BC_OUTFLOW && p->bc[d] != RGRMHD_BC_EXTERNAL) return RGRMHD_E_INVALID;
    if (p->bc[d] == RGRMHD_BC_EXTERNAL && (p->n[d] < 3 || p->charge_mode == RGRMHD_CHARGE_DIV_E)) return RGRMHD_E_INVALID;
  }
  if (p->sigma_model < RGRMHD_SIGMA_UNIFORM || p->sigma_model > RGRMHD_SIGMA_ATMO) return RGRMHD_E_INVALID;
  if (p->charge_mode != RGRMHD_CHARGE_FACE_OHM && p->charge_mode != RGRMHD_CHARGE_CELL_CURRENT &&
      p->charge_mode != RGRMHD_CHARGE_DIV_E)
    return RGRMHD_E_INVALID;
  if (p->sigma_model == RGRMHD_SIGMA_POWER_D &&
      (p->sigma_exp < 0.0 || std::fabs(p->sigma_exp - std::lround(p->sigma_exp)) > 0.0 || !(p->sigma_dref > 0.0)))
    return RGRMHD_E_INVALID;
  if (p->wave_speed_mode != RGRMHD_WAVE_LIGHT && p->wave_speed_mode != RGRMHD_WAVE_MHD_INSIDE) return RGRMHD_E_INVALID;
  if (p->weno_eps > 0.0 && p->weno_eps < 1e-60) return RGRMHD_E_INVALID;   // product-form weights would underflow
  if (p->rho_floor < 0.0 || !(p->kappa == p->kappa)) return RGRMHD_E_INVALID;

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || p->device < 0 || p->device >= ndev) {
    cudaGetLastError();
    return RGRMHD_E_CUDA;
  }
  rgrmhd_s* h = new (std::nothrow) rgrmhd_s();
  if (!h) return RGRMHD_E_NOMEM;
  h->par = *p;
  h->device = p->device;
  DeviceGuard guard(h->device);
  if (!guard.ok) { delete h; return RGRMHD_E_CUDA; }

  rg::GridView& G = h->G;
  std::memset(&G, 0, sizeof(G));
  G.ntot = 1;
  for (int d = 0; d < 3; ++d) {
    G.n[d] = p->n[d];
    G.g[d] = p->n[d] > 1 ? 3 : 0;
    G.np[d] = p->n[d] + 2 * G.g[d];
    G.bc[d] = p->bc[d];
    G.dx[d] = p->dx[d];
    G.inv_dx[d] = p->n[d] > 1 ? 1.0 / p->dx[d] : 0.0;
    G.inv_12dx[d] = p->n[d] > 1 ? 1.0 / (12.0 * p->dx[d]) : 0.0;
    G.ntot *= G.np[d];
  }
  G.stride[0] = 1; G.stride[1] = G.np[0]; G.stride[2] = (long long)G.np[0] * G.np[1];
  G.Gamma = p->gamma_eos;
  G.gog1 = p->gamma_eos / (p->gamma_eos - 1.0);
  G.gm1og = (p->gamma_eos - 1.0) / p->gamma_eos;
  G.sigma_model = p->sigma_model; G.sigma0 = p->sigma0; G.sigma_dref = p->sigma_dref;
  G.sigma_exp = (int)std::lround(p->sigma_exp);
  G.kappa = p->kappa;
  G.rho_floor = p->rho_floor;
  G.p_atmo = p->rho_floor > 0.0 ? p->k_atmo * std::pow(p->rho_floor, p->gamma_eos) : 0.0;   // p = K rho^Gamma
  G.tol = p->c2p_tol > 0.0 ? p->c2p_tol : 8.0 * std::ldexp(1.0, -52);
  G.maxit = p->c2p_max_iter > 0 ? p->c2p_max_iter : 100;
  G.charge_mode = p->charge_mode;
  G.wave_mode = p->wave_speed_mode; G.wave_rho_switch = p->wave_rho_switch;
  G.weno_eps = p->weno_eps > 0.0 ? p->weno_eps : 1e-26;

  const int nfields = rg::NMET + 1 + rg::NPRIM + 3 + rg::NCONS + rg::NCONS + 3 + rg::NCONS;   // + the static source fields: set_metric
  h->field_stride = (G.ntot + 31) / 32 * 32;
  const size_t bytes = (size_t)nfields * (size_t)h->field_stride * sizeof(double);
  cudaError_t e = cudaMalloc((void**)&h->slab, bytes);
  if (e != cudaSuccess) { cudaGetLastError(); delete h; return RGRMHD_E_NOMEM; }
  e = cudaMalloc((void**)&h->stats_dev, sizeof(rg::StatsDev) + 2 * sizeof(unsigned long long));
  if (e != cudaSuccess) { cudaGetLastError(); cudaFree(h->slab); delete h; return RGRMHD_E_NOMEM; }
  h->maxspeed_dev = (unsigned long long*)(h->stats_dev + 1);
  e = cudaMemset(h->slab, 0, bytes);
  if (e == cudaSuccess) e = cudaMemset(h->stats_dev, 0, sizeof(rg::StatsDev) + 2 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, h->device);
  if (e != cudaSuccess) { cudaGetLastError(); cudaFree(h->slab); cudaFree(h->stats_dev); delete h; return RGRMHD_E_CUDA; }
  G.src_mask = h->maxspeed_dev + 1;
  G.maxspeed_word = h->maxspeed_dev;
  double* q = h->slab;
  auto next = [&]() { double* r = q; q += h->field_stride; return r; };
  for (int v = 0; v < rg::NMET; ++v) G.met[v] = next();
  { double* s = next(); G.sigma = (p->sigma_model == RGRMHD_SIGMA_ARRAY) ? s : nullptr; }
  for (int v = 0; v < rg::NPRIM; ++v) G.P[v] = next();
  for (int v = 0; v < 3; ++v) G.jc[v] = next();
  for (int v = 0; v < rg::NCONS; ++v) G.Un[v] = next();
  for (int v = 0; v < rg::NCONS; ++v) G.Us[v] = next();
  for (int v = 0; v < 3; ++v) G.X1[v] = next();
  for (int v = 0; v < rg::NSRC; ++v) G.src[v] = nullptr;   // allocated by set_metric
  for (int v = 0; v < rg::NCONS; ++v) G.dU[v] = next();
  e = cudaDeviceSynchronize();
  if (e != cudaSuccess) { cudaFree(h->slab); cudaFree(h->stats_dev); delete h; return RGRMHD_E_CUDA; }
  h->tma = rg::tma_create(G);
  *out = h;
  return RGRMHD_OK;
}

int rgrmhd_destroy(rgrmhd_t h) {
  if (!h) return RGRMHD_E_INVALID;
  {
    DeviceGuard guard(h->device);
    cudaStreamSynchronize(h->stream);
    for (auto& t : h->timed) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); }
    cudaFree(h->slab);
    cudaFree(h->slab2);
    cudaFree(h->slab_src);
    cudaFree(h->stats_dev);
    rg::tma_destroy(h->tma);
  }
  delete h;
  return RGRMHD_OK;
}

// optional per-kernel event bracket (rgrmhd_set_timing)
static const size_t kMaxTimed = 1 << 16;
static cudaError_t timed(rgrmhd_t h, int cls, const std::function<cudaError_t()>& launch) {
  if (!h->timing) return launch();
  rgrmhd_s::Timed t{cls, nullptr, nullptr};
  cudaError_t e = cudaEventCreate(&t.a);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&t.b);
  if (e != cudaSuccess) { cudaEventDestroy(t.a); return e; }
  e = cudaEventRecord(t.a, h->stream);
  if (e == cudaSuccess) e = launch();
  if (e == cudaSuccess) e = cudaEventRecord(t.b, h->stream);
  if (e != cudaSuccess) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); return e; }
  if (h->timed.size() >= kMaxTimed) {   // nobody collects them (rgrmhd_get_timing): drop the oldest bracket
    cudaEventDestroy(h->timed.front().a); cudaEventDestroy(h->timed.front().b);
    h->timed.erase(h->timed.begin());
  }
  h->timed.push_back(t);
  return e;
}

// rgrmhd_step leaves the recovery of its new state (reading R12) to whoever needs that state next: the next step
// runs it inside its first recovery kernel (k_c2p<4>), every other entry point that reads or replaces the state
// launches it here first.
static int finish_step(rgrmhd_t h) {
  if (h->poisoned || h->part != 0) return RGRMHD_E_STATE;   // (a split step must be completed first)
  if (!h->pending_final) return RGRMHD_OK;
  DeviceGuard guard(h->device);
  const bool fuse_cfl = h->G.wave_mode == rg::WAVE_MHD_INSIDE;
  if (fuse_cfl) RG_CUDA(h, cudaMemsetAsync(h->maxspeed_dev, 0, sizeof(unsigned long long), h->stream));
  const cudaError_t e = timed(h, RGRMHD_K_C2P, [&] { return rg::launch_c2p(h->G, 3, 0.0, h->stats_dev, h->stream); });
  if (e != cudaSuccess) { h->poisoned = true; return fail_cuda(h, e, "launch_c2p(final recovery)"); }
  ++h->launches;
  h->pending_final = false;
  h->maxspeed_fused = fuse_cfl;
  return RGRMHD_OK;
}

// charge mode DIV_E: q and calQ of the new state from its electric field, when somebody reads the state
static int finish_charge(rgrmhd_t h) {
  if (!h->charge_final_due) return RGRMHD_OK;
  const rg::GridView& G = h->G;
  if (G.n[0] > 1 || G.n[1] > 1 || G.n[2] > 1) {
    RG_CUDA(h, rg::launch_ghost_fill(G, G.P + rg::EX, 3, h->stream));
    ++h->launches;
  }
  RG_CUDA(h, rg::launch_charge_div_e(G, 3, 0.0, h->stream));
  ++h->launches;
  h->charge_final_due = false;
  return RGRMHD_OK;
}

int rgrmhd_flush(rgrmhd_t h) {
  if (!h) return RGRMHD_E_INVALID;
  return finish_step(h);
}

int rgrmhd_set_stream(rgrmhd_t h, void* cuda_stream) {
  if (!h) return RGRMHD_E_INVALID;
  DeviceGuard guard(h->device);
  int rc;
  if (!h->poisoned && (rc = finish_step(h))) return rc;   // on the stream the step was enqueued on
  const cudaStream_t next = (cudaStream_t)cuda_stream;
  if (next != h->stream) {
    // everything already enqueued on the old stream (copies of set_*, kernels, the recovery just flushed) must be
    // complete before later work on the new stream touches the state: event on the old, wait on the new
    cudaEvent_t ev;
    RG_CUDA(h, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    cudaError_t e = cudaEventRecord(ev, h->stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(next, ev, 0);
    cudaEventDestroy(ev);                                  // released once the recorded work has completed
    if (e != cudaSuccess) return fail_cuda(h, e, "stream hand-over");
    h->stream = next;
  }
  return RGRMHD_OK;
}

int rgrmhd_set_rhs_variant(rgrmhd_t h, int variant) {
  if (!h || variant < 0 || variant > 2) return RGRMHD_E_INVALID;
  h->rhs_variant = variant;
  return RGRMHD_OK;
}

int rgrmhd_get_rhs_variant(rgrmhd_t h, int* host_out) {
  if (!h || !host_out) return RGRMHD_E_INVALID;
  if (h->last_rhs_variant >= 0) { *host_out = h->last_rhs_variant; return RGRMHD_OK; }
  const bool tma = h->rhs_variant == 0 && h->tma != nullptr;
  *host_out = tma ? 0 : (h->rhs_variant != 1 && rg::rhs_pencil_supported(h->G)) ? 2 : 1;
  return RGRMHD_OK;
}

static int copy_in(rgrmhd_t h, const double* dst_dev, const double* src) {
  RG_CUDA(h, cudaMemcpyAsync((void*)dst_dev, src, (size_t)h->G.ntot * sizeof(double), cudaMemcpyDefault, h->stream));
  return RGRMHD_OK;
}
static int copy_out(rgrmhd_t h, double* dst, const double* src_dev) {
  RG_CUDA(h, cudaMemcpyAsync(dst, src_dev, (size_t)h->G.ntot * sizeof(double), cudaMemcpyDefault, h->stream));
  return RGRMHD_OK;
}

int rgrmhd_set_metric(rgrmhd_t h, const double* alpha, const double* const beta[3], const double* const gam[6],
                      const double* const K[6]) {
  if (!h || !alpha || !beta || !gam || !K) return RGRMHD_E_INVALID;
  for (int i = 0; i < 3; ++i) if (!beta[i]) return RGRMHD_E_INVALID;
  for (int i = 0; i < 6; ++i) if (!gam[i] || !K[i]) return RGRMHD_E_INVALID;
  DeviceGuard guard(h->device);
  int rc;
  if ((rc = finish_step(h))) return rc;
  if ((rc = copy_in(h, h->G.met[rg::MALP], alpha))) return rc;
  for (int i = 0; i < 3; ++i) if ((rc = copy_in(h, h->G.met[rg::MBX + i], beta[i]))) return rc;
  for (int i = 0; i < 6; ++i) {
    if ((rc = copy_in(h, h->G.met[rg::MGXX + i], gam[i]))) return rc;
    if ((rc = copy_in(h, h->G.met[rg::MKXX + i], K[i]))) return rc;
  }
  h->maxspeed_cached = false; h->maxspeed_fused = false;
  // static source coefficients (rgrmhd_sources.cuh): find the fields that are not identically zero, allocate those, fill them
  RG_CUDA(h, rg::launch_metric_coeffs(h->G, false, h->stream));
  unsigned long long mask = 0;
  RG_CUDA(h, cudaMemcpyAsync(&mask, h->G.src_mask, sizeof(mask), cudaMemcpyDeviceToHost, h->stream));
  RG_CUDA(h, cudaStreamSynchronize(h->stream));
  int nsrc = 0;
  for (int q = 0; q < rg::NSRC; ++q) nsrc += (int)((mask >> q) & 1ull);
  if (nsrc != h->nsrc_fields || !h->slab_src) {
    cudaFree(h->slab_src);
    h->slab_src = nullptr; h->nsrc_fields = 0;
    if (nsrc > 0 && cudaMalloc((void**)&h->slab_src, (size_t)nsrc * (size_t)h->field_stride * sizeof(double)) != cudaSuccess) {
      cudaGetLastError();
      h->have_metric = false;
      return RGRMHD_E_NOMEM;
    }
    h->nsrc_fields = nsrc;
  }
  {
    double* q0 = h->slab_src;
    for (int q = 0; q < rg::NSRC; ++q) {
      if ((mask >> q) & 1ull) { h->G.src[q] = q0; q0 += h->field_stride; } else h->G.src[q] = nullptr;
    }
  }
  RG_CUDA(h, rg::launch_metric_coeffs(h->G, true, h->stream));
  h->launches += 2;
  h->have_metric = true;
  return RGRMHD_OK;
}

int rgrmhd_set_sigma(rgrmhd_t h, const double* sigma) {
  if (!h || !sigma) return RGRMHD_E_INVALID;
  if (h->par.sigma_model != RGRMHD_SIGMA_ARRAY) return RGRMHD_E_STATE;
  DeviceGuard guard(h->device);
  int rc;
  if ((rc = finish_step(h))) return rc;
  if ((rc = copy_in(h, h->G.sigma, sigma))) return rc;
  h->have_sigma = true;
  return RGRMHD_OK;
}

int rgrmhd_set_prims(rgrmhd_t h, const double* const prims[14]) {
  if (!h || !prims) return RGRMHD_E_INVALID;
  for (int v = 0; v < rg::NPRIM; ++v) if (!prims[v]) return RGRMHD_E_INVALID;
  if (!h->have_metric) return RGRMHD_E_STATE;
  DeviceGuard guard(h->device);
  int rc;
  if (h->poisoned) { h->poisoned = false; h->pending_final = false; }
  h->part = 0;   // the half-advanced state is replaced below
  if ((rc = finish_step(h))) return rc;   // keeps the statistics complete; the state itself is replaced
  for (int v = 0; v < rg::NPRIM; ++v) if ((rc = copy_in(h, h->G.P[v], prims[v]))) return rc;
  for (int q = 0; q < 3; ++q)
    RG_CUDA(h, cudaMemsetAsync(h->G.jc[q], 0, (size_t)h->G.ntot * sizeof(double), h->stream));
  RG_CUDA(h, rg::launch_prim2cons(h->G, h->stream));
  ++h->launches;
  h->have_prims = true;
  h->charge_final_due = false;
  h->maxspeed_fused = false;
  return RGRMHD_OK;
}

// ---- general IMEX-RK driver (Eq. 32-34) ---------------------------------
namespace {
struct Tableau { int s; double At[4][4], wt[4], A[4][4], w[4]; };

// The schemes the paper incorporates.  PAPER.md prints only Table I's scheme (through Eq. 35-37); the
// others are the published Pareschi-Russo tableaux, checked against the IMEX order conditions by the tests.
bool tableau_of(int time_scheme, Tableau& T) {
  std::memset(&T, 0, sizeof(T));
  const double g = 1.0 - 1.0 / std::sqrt(2.0);
  switch (time_scheme) {
    case RGRMHD_TIME_IMEX_SSP2_222_GENERAL:
      T.s = 2;
      T.At[1][0] = 1.0; T.wt[0] = T.wt[1] = 0.5;
      T.A[0][0] = g; T.A[1][0] = 1.0 - 2.0 * g; T.A[1][1] = g; T.w[0] = T.w[1] = 0.5;
      return true;
    case RGRMHD_TIME_IMEX_SSP2_332:
      T.s = 3;
      T.At[1][0] = 0.5; T.At[2][0] = 0.5; T.At[2][1] = 0.5; T.wt[0] = T.wt[1] = T.wt[2] = 1.0 / 3.0;
      T.A[0][0] = 0.25; T.A[1][1] = 0.25; T.A[2][0] = T.A[2][1] = T.A[2][2] = 1.0 / 3.0;
      T.w[0] = T.w[1] = T.w[2] = 1.0 / 3.0;
      return true;
    case RGRMHD_TIME_IMEX_SSP3_332:
      T.s = 3;
      T.At[1][0] = 1.0; T.At[2][0] = 0.25; T.At[2][1] = 0.25; T.wt[0] = T.wt[1] = 1.0 / 6.0; T.wt[2] = 2.0 / 3.0;
      T.A[0][0] = g; T.A[1][0] = 1.0 - 2.0 * g; T.A[1][1] = g; T.A[2][0] = 0.5 - g; T.A[2][2] = g;
      T.w[0] = T.w[1] = 1.0 / 6.0; T.w[2] = 2.0 / 3.0;
      return true;
    case RGRMHD_TIME_IMEX_SSP3_433: {
      const double al = 0.24169426078821, be = 0.06042356519705, et = 0.12915286960590;
      T.s = 4;
      T.At[2][1] = 1.0; T.At[3][1] = 0.25; T.At[3][2] = 0.25; T.wt[1] = T.wt[2] = 1.0 / 6.0; T.wt[3] = 2.0 / 3.0;
      T.A[0][0] = al; T.A[1][0] = -al; T.A[1][1] = al; T.A[2][1] = 1.0 - al; T.A[2][2] = al;
      T.A[3][0] = be; T.A[3][1] = et; T.A[3][2] = 0.5 - be - et - al; T.A[3][3] = al;
      T.w[1] = T.w[2] = 1.0 / 6.0; T.w[3] = 2.0 / 3.0;
      return true;
    }
  }
  return false;
}
}  // namespace

static int step_general(rgrmhd_t h, double dt, int recon, const Tableau& T) {
  DeviceGuard guard(h->device);
  const rg::GridView& G = h->G;
  cudaStream_t st = h->stream;
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  int rc;
  if ((rc = finish_step(h))) return rc;                       // a deferred recovery of the SSP2(2,2,2) path, if any
  if (T.s > 2 && !h->slab2) {                                 // accumulators of stages 2 and 3
    const size_t bytes = (size_t)2 * rg::NCONS * (size_t)h->field_stride * sizeof(double);
    if (cudaMalloc((void**)&h->slab2, bytes) != cudaSuccess) { cudaGetLastError(); h->slab2 = nullptr; return RGRMHD_E_NOMEM; }
  }
  rg::StageGen W;
  std::memset(&W, 0, sizeof(W));
  W.nstages = T.s;
  for (int v = 0; v < rg::NCONS; ++v) {
    W.acc[4].f[v] = G.Un[v];
    W.acc[1].f[v] = G.Us[v];
    W.acc[2].f[v] = h->slab2 ? h->slab2 + (size_t)v * h->field_stride : nullptr;
    W.acc[3].f[v] = h->slab2 ? h->slab2 + (size_t)(rg::NCONS + v) * h->field_stride : nullptr;
    W.acc[0].f[v] = G.Un[v];                                  // never used as a target
  }
  double* ghost_fields[rg::NPRIM + 3];
  for (int v = 0; v < rg::NPRIM; ++v) ghost_fields[v] = G.P[v];
  for (int q = 0; q < 3; ++q) ghost_fields[rg::NPRIM + q] = G.jc[q];
  const int nghost_fields = rg::NPRIM + (G.charge_mode != rg::CHARGE_FACE_OHM ? 3 : 0);
  const bool div_e = G.charge_mode == rg::CHARGE_DIV_E;
  const bool any_active = G.n[0] > 1 || G.n[1] > 1 || G.n[2] > 1;
  const bool tma = h->rhs_variant == 0 && h->tma != nullptr;
  const bool pencil = !tma && h->rhs_variant != 1 && rg::rhs_pencil_supported(G);
  h->last_rhs_variant = tma ? 0 : pencil ? 2 : 1;
#define RG_STEP(call)                                                              \
  do {                                                                             \
    cudaError_t e__ = (call);                                                      \
    if (e__ != cudaSuccess) { h->poisoned = true; h->pending_final = false; return fail_cuda(h, e__, #call); } \
  } while (0)
  h->maxspeed_fused = false;
  bool have_d = false;                                        // G.dU holds dt (-div F) of the previous stage
  for (int i = 0; i <= T.s; ++i) {
    const bool final = i == T.s;
    W.stage = i;
    W.init = (i == 0);
    W.use_dprev = have_d ? 1 : 0;
    W.aii = final ? 0.0 : T.A[i][i];
    for (int slot = 0; slot < 5; ++slot) {
      const int tgt = slot == 4 ? T.s : slot;                 // row of the tableau; row s = the weights
      auto at = [&](int row, int col) { return col < 0 ? 0.0 : row == T.s ? T.wt[col] : T.At[row][col]; };
      auto ai = [&](int row, int col) { return row == T.s ? T.w[col] : T.A[row][col]; };
      W.w_dprev[slot] = (have_d && tgt >= i && slot < 5 && (slot == 4 || slot < T.s)) ? at(tgt, i - 1) : 0.0;
      W.w_src[slot] = (!final && tgt > i && (slot == 4 || slot < T.s)) ? at(tgt, i) : 0.0;
      W.w_stiff[slot] = (!final && tgt > i && (slot == 4 || slot < T.s)) ? ai(tgt, i) / T.A[i][i] : 0.0;
    }
    RG_STEP(timed(h, RGRMHD_K_C2P, [&] { return rg::launch_stage_gen(G, W, dt, h->stats_dev, st); }));
    ++h->launches;
    if (final) break;
    bool used = T.wt[i] != 0.0;
    for (int k = i + 1; k < T.s; ++k) used = used || T.At[k][i] != 0.0;
    have_d = used;
    if (!used) continue;                                      // nobody needs F of this stage (SSP3(4,3,3), stage 1)
    if (any_active) { RG_STEP(timed(h, RGRMHD_K_GHOST, [&] { return rg::launch_ghost_fill(G, ghost_fields, nghost_fields, st); })); ++h->launches; }
    if (div_e) {
      RG_STEP(timed(h, RGRMHD_K_GHOST, [&] { return rg::launch_charge_div_e(G, 0, dt, st); }));
      RG_STEP(timed(h, RGRMHD_K_GHOST, [&] { return rg::launch_charge_sources_gen(G, W, dt, st); }));
      h->launches += 2;
    }
    RG_STEP(timed(h, RGRMHD_K_RHS, [&] {
      return tma    ? rg::launch_rhs_tma(G, h->tma, dt, 1, recon, h->sm_count, st)
           : pencil ? rg::launch_rhs_pencil(G, dt, 1, recon, h->sm_count, st)
                    : rg::launch_rhs_simple(G, dt, 1, recon, st);
    }));                                                      // stage-1 flavour: writes dU = dt (-div F)
    ++h->launches;
  }
#undef RG_STEP
  h->pending_final = false;
  h->charge_final_due = div_e;
  h->solves += (T.s + 1) * nint;
  return RGRMHD_OK;
}

// One IMEX-SSP2(2,2,2) step in three parts (Eq. 35-37); rgrmhd_step runs them back to back.
//   part 0: recovery of stage 1 (+ the pending final recovery of the previous step) and its ghost fill
//   part 1: flux divergence of stage 1, recovery of stage 2 and its ghost fill
//   part 2: flux divergence of stage 2 (the final recovery stays deferred, see finish_step)
static int step222_part(rgrmhd_t h, int part) {
  DeviceGuard guard(h->device);
  const rg::GridView& G = h->G;
  cudaStream_t st = h->stream;
  const double dt = h->cur_dt;
  const int recon = h->cur_recon;
  const long long nint = (long long)G.n[0] * G.n[1] * G.n[2];
  double* ghost_fields[rg::NPRIM + 3];
  for (int v = 0; v < rg::NPRIM; ++v) ghost_fields[v] = G.P[v];
  for (int q = 0; q < 3; ++q) ghost_fields[rg::NPRIM + q] = G.jc[q];
  const int nghost_fields = rg::NPRIM + (G.charge_mode != rg::CHARGE_FACE_OHM ? 3 : 0);
  const bool div_e = G.charge_mode == rg::CHARGE_DIV_E;
  const bool any_active = G.n[0] > 1 || G.n[1] > 1 || G.n[2] > 1;
  const bool tma = h->rhs_variant == 0 && h->tma != nullptr;
  const bool pencil = !tma && h->rhs_variant != 1 && rg::rhs_pencil_supported(G);
  auto rhs = [&](int stage) {
    return tma    ? rg::launch_rhs_tma(G, h->tma, dt, stage, recon, h->sm_count, st)
         : pencil ? rg::launch_rhs_pencil(G, dt, stage, recon, h->sm_count, st)
                  : rg::launch_rhs_simple(G, dt, stage, recon, st);
  };
  h->last_rhs_variant = tma ? 0 : pencil ? 2 : 1;
  // From the first launch on the state is in flight: if any launch fails, the handle is marked poisoned and every
  // later call but set_prims / destroy returns RGRMHD_E_STATE (the state is half advanced, nothing can read it safely).
#define RG_STEP(call)                                                              \
  do {                                                                             \
    cudaError_t e__ = (call);                                                      \
    if (e__ != cudaSuccess) { h->poisoned = true; h->pending_final = false; h->part = 0; return fail_cuda(h, e__, #call); } \
  } while (0)
  h->maxspeed_fused = false;
  if (part == 0) {
    // stage 1 (Eq. 35): X*1 = X^n, Y1 = Y^n.  The recovery kernel also applies the point-wise half of the
    // right-hand side (sources, implicit terms) to the stage target; the flux kernel adds -w dt div F.
    // (if the previous step's final recovery is still due, the same kernel runs it first: k_c2p<4>)
    const int first = h->pending_final ? 4 : 1;
    RG_STEP(timed(h, RGRMHD_K_C2P, [&] { return rg::launch_c2p(G, first, dt, h->stats_dev, st); }));
    h->pending_final = false;
    if (any_active) RG_STEP(timed(h, RGRMHD_K_GHOST, [&] { return rg::launch_ghost_fill(G, ghost_fields, nghost_fields, st); }));
    h->launches += 1 + (any_active ? 1 : 0);
  } else if (part == 1) {
    if (div_e) RG_STEP(timed(h, RGRMHD_K_GHOST, [&] { return rg::launch_charge_div_e(G, 1, dt, st); }));
    RG_STEP(timed(h, RGRMHD_K_RHS, [&] { return rhs(1); }));   // -> U*2 (Eq. 36)
    // stage 2 (Eq. 36)
    RG_STEP(timed(h, RGRMHD_K_C2P, [&] { return rg::launch_c2p(G, 2, dt, h->stats_dev, st); }));
    if (any_active) RG_STEP(timed(h, RGRMHD_K_GHOST, [&] { return rg::launch_ghost_fill(G, ghost_fields, nghost_fields, st); }));
    h->launches += 2 + (any_active ? 1 : 0) + (div_e ? 1 : 0);
  } else {
    if (div_e) RG_STEP(timed(h, RGRMHD_K_GHOST, [&] { return rg::launch_charge_div_e(G, 2, dt, st); }));
    RG_STEP(timed(h, RGRMHD_K_RHS, [&] { return rhs(2); }));   // -> U^{n+1} (Eq. 37)
    // recovery of the new state at fixed calE (reading R12): deferred, see finish_step
    h->pending_final = true;
    h->charge_final_due = div_e;
    h->solves += 3 * nint;
    h->launches += 1 + (div_e ? 1 : 0);
  }
#undef RG_STEP
  return RGRMHD_OK;
}

int rgrmhd_step(rgrmhd_t h, double dt, int scheme) {
  if (!h || !(dt > 0.0)) return RGRMHD_E_INVALID;
  const int recon = scheme & RGRMHD_RECON_MASK;
  const int time_scheme = scheme & ~RGRMHD_RECON_MASK;
  Tableau T;
  if (recon > RGRMHD_RECON_WENO5 || (time_scheme != RGRMHD_TIME_IMEX_SSP2_222 && !tableau_of(time_scheme, T)))
    return RGRMHD_E_INVALID;
  if (!h->have_metric || !h->have_prims || (h->par.sigma_model == RGRMHD_SIGMA_ARRAY && !h->have_sigma) || h->poisoned)
    return RGRMHD_E_STATE;
  if (time_scheme != RGRMHD_TIME_IMEX_SSP2_222) {
    for (int d = 0; d < 3; ++d) if (h->G.bc[d] == rg::BC_EXTERNAL) return RGRMHD_E_INVALID;   // no exchange points inside
    return step_general(h, dt, recon, T);
  }
  if (h->part != 0) return RGRMHD_E_STATE;               // a split step (rgrmhd_step_begin) is in flight
  for (int d = 0; d < 3; ++d) if (h->G.bc[d] == rg::BC_EXTERNAL) return RGRMHD_E_INVALID;     // needs the split form
  h->cur_dt = dt; h->cur_recon = recon;
  int rc;
  for (int part = 0; part < 3; ++part) if ((rc = step222_part(h, part))) return rc;
  return RGRMHD_OK;
}

// ---- the same step in three parts, for callers that own ghost layers (bc = RGRMHD_BC_EXTERNAL: a slab of a larger
// grid): after rgrmhd_step_begin and after the first rgrmhd_step_continue the stage's
// primitives and conduction current are complete in the interior and in the ghost layers the library fills itself;
// the caller exchanges the external layers (rgrmhd_halo_pack / rgrmhd_halo_unpack) and continues.
int rgrmhd_step_begin(rgrmhd_t h, double dt, int scheme) {
  if (!h || !(dt > 0.0)) return RGRMHD_E_INVALID;
  const int recon = scheme & RGRMHD_RECON_MASK;
  if (recon > RGRMHD_RECON_WENO5 || (scheme & ~RGRMHD_RECON_MASK) != RGRMHD_TIME_IMEX_SSP2_222) return RGRMHD_E_INVALID;
  if (!h->have_metric || !h->have_prims || (h->par.sigma_model == RGRMHD_SIGMA_ARRAY && !h->have_sigma) || h->poisoned ||
      h->part != 0)
    return RGRMHD_E_STATE;
  h->cur_dt = dt; h->cur_recon = recon;
  const int rc = step222_part(h, 0);
  if (rc == RGRMHD_OK) h->part = 1;
  return rc;
}

int rgrmhd_step_continue(rgrmhd_t h, int* more) {
  if (!h || !more) return RGRMHD_E_INVALID;
  if (h->part != 1 && h->part != 2) return RGRMHD_E_STATE;
  if (h->poisoned) return RGRMHD_E_STATE;
  const int rc = step222_part(h, h->part);
  if (rc != RGRMHD_OK) { h->part = 0; return rc; }
  h->part = (h->part == 1) ? 2 : 0;
  *more = h->part != 0;
  return RGRMHD_OK;
}

// ---- halo layers of the stage primitives and of the conduction current (17 fields), SURVEY.md Sec. 8(e) ------------
int rgrmhd_halo_doubles(rgrmhd_t h, int dir, long long* host_out) {
  if (!h || !host_out || dir < 0 || dir > 2 || h->G.n[dir] < 3) return RGRMHD_E_INVALID;
  long long plane = 1;
  for (int d = 0; d < 3; ++d) if (d != dir) plane *= h->G.np[d];
  *host_out = (long long)(rg::NPRIM + 3) * 3 * plane;
  return RGRMHD_OK;
}

static int halo_copy(rgrmhd_t h, int dir, int side, double* buf, bool pack) {
  if (!h || !buf || dir < 0 || dir > 2 || (side != 0 && side != 1) || h->G.n[dir] < 3) return RGRMHD_E_INVALID;
  if (!h->have_prims || h->poisoned) return RGRMHD_E_STATE;
  DeviceGuard guard(h->device);
  double* fields[rg::NPRIM + 3];
  for (int v = 0; v < rg::NPRIM; ++v) fields[v] = h->G.P[v];
  for (int q = 0; q < 3; ++q) fields[rg::NPRIM + q] = h->G.jc[q];
  RG_CUDA(h, rg::launch_halo_copy(h->G, fields, rg::NPRIM + 3, dir, side, buf, pack, h->stream));
  ++h->launches;
  return RGRMHD_OK;
}
int rgrmhd_halo_pack(rgrmhd_t h, int dir, int side, double* dev_buf) { return halo_copy(h, dir, side, dev_buf, true); }
int rgrmhd_halo_unpack(rgrmhd_t h, int dir, int side, const double* dev_buf) {
  return halo_copy(h, dir, side, const_cast<double*>(dev_buf), false);
}

int rgrmhd_max_speed(rgrmhd_t h, double* host_out) {
  if (!h || !host_out) return RGRMHD_E_INVALID;
  if (!h->have_metric) return RGRMHD_E_STATE;
  DeviceGuard guard(h->device);
  if (h->G.wave_mode == rg::WAVE_LIGHT && h->maxspeed_cached) { *host_out = h->maxspeed_value; return RGRMHD_OK; }
  if (h->G.wave_mode == rg::WAVE_MHD_INSIDE && h->have_prims) {   // state dependent: needs the current primitives
    int rc;
    if ((rc = finish_step(h))) return rc;
  }
  if (!(h->G.wave_mode == rg::WAVE_MHD_INSIDE && h->maxspeed_fused)) {   // else: the final recovery has just reduced it
    RG_CUDA(h, cudaMemsetAsync(h->maxspeed_dev, 0, sizeof(unsigned long long), h->stream));
    RG_CUDA(h, rg::launch_max_speed(h->G, h->maxspeed_dev, h->have_prims, h->sm_count, h->stream));
    ++h->launches;
  }
  unsigned long long bits = 0;
  RG_CUDA(h, cudaMemcpyAsync(&bits, h->maxspeed_dev, sizeof(bits), cudaMemcpyDeviceToHost, h->stream));
  RG_CUDA(h, cudaStreamSynchronize(h->stream));
  double v;
  std::memcpy(&v, &bits, sizeof(v));
  *host_out = v;
  if (h->G.wave_mode == rg::WAVE_LIGHT) { h->maxspeed_cached = true; h->maxspeed_value = v; }
  return RGRMHD_OK;
}

int rgrmhd_get_prims(rgrmhd_t h, double* const prims[14]) {
  if (!h || !prims) return RGRMHD_E_INVALID;
  for (int v = 0; v < rg::NPRIM; ++v) if (!prims[v]) return RGRMHD_E_INVALID;
  if (!h->have_prims) return RGRMHD_E_STATE;
  DeviceGuard guard(h->device);
  int rc;
  if ((rc = finish_step(h))) return rc;
  if ((rc = finish_charge(h))) return rc;
  const rg::GridView& G = h->G;
  if (G.n[0] > 1 || G.n[1] > 1 || G.n[2] > 1) {
    RG_CUDA(h, rg::launch_ghost_fill(G, G.P, rg::NPRIM, h->stream));
    ++h->launches;
  }
  for (int v = 0; v < rg::NPRIM; ++v) if ((rc = copy_out(h, prims[v], G.P[v]))) return rc;
  return RGRMHD_OK;
}

int rgrmhd_get_cons(rgrmhd_t h, double* const cons[14]) {
  if (!h || !cons) return RGRMHD_E_INVALID;
  for (int v = 0; v < rg::NCONS; ++v) if (!cons[v]) return RGRMHD_E_INVALID;
  if (!h->have_prims) return RGRMHD_E_STATE;
  DeviceGuard guard(h->device);
  int rc;
  if ((rc = finish_step(h))) return rc;
  if ((rc = finish_charge(h))) return rc;
  for (int v = 0; v < rg::NCONS; ++v) if ((rc = copy_out(h, cons[v], h->G.Un[v]))) return rc;
  return RGRMHD_OK;
}

int rgrmhd_get_stats(rgrmhd_t h, rgrmhd_stats* host_out) {
  if (!h || !host_out) return RGRMHD_E_INVALID;
  DeviceGuard guard(h->device);
  int rc;
  if ((rc = finish_step(h))) return rc;
  rg::StatsDev s;
  RG_CUDA(h, cudaMemcpyAsync(&s, h->stats_dev, sizeof(s), cudaMemcpyDeviceToHost, h->stream));
  RG_CUDA(h, cudaStreamSynchronize(h->stream));
  host_out->c2p_solves = h->solves;
  host_out->c2p_evals = (long long)s.evals;
  host_out->c2p_failures = (long long)s.failures;
  host_out->floor_resets = (long long)s.floors;
  host_out->c2p_max_evals = s.max_evals;
  host_out->reserved = 0;
  return RGRMHD_OK;
}

int rgrmhd_reset_stats(rgrmhd_t h) {
  if (!h) return RGRMHD_E_INVALID;
  DeviceGuard guard(h->device);
  int rc;
  if ((rc = finish_step(h))) return rc;
  RG_CUDA(h, cudaMemsetAsync(h->stats_dev, 0, sizeof(rg::StatsDev), h->stream));
  h->solves = 0;
  return RGRMHD_OK;
}

int rgrmhd_set_timing(rgrmhd_t h, int enable) {
  if (!h) return RGRMHD_E_INVALID;
  h->timing = enable != 0;
  return RGRMHD_OK;
}

int rgrmhd_get_timing(rgrmhd_t h, double ms[RGRMHD_K_COUNT], long long launches[RGRMHD_K_COUNT]) {
  if (!h || !ms || !launches) return RGRMHD_E_INVALID;
  DeviceGuard guard(h->device);
  for (int k = 0; k < RGRMHD_K_COUNT; ++k) { ms[k] = 0.0; launches[k] = 0; }
  int rc;
  if ((rc = finish_step(h))) return rc;
  RG_CUDA(h, cudaStreamSynchronize(h->stream));
  for (auto& t : h->timed) {
    float f = 0.f;
    if (cudaEventElapsedTime(&f, t.a, t.b) == cudaSuccess) { ms[t.cls] += f; launches[t.cls] += 1; }
    cudaEventDestroy(t.a); cudaEventDestroy(t.b);
  }
  h->timed.clear();
  return RGRMHD_OK;
}

namespace {
__global__ void __launch_bounds__(256) k_dfma_peak(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 12345.678) out[0] = s;   // never true for the arguments used; keeps the chains alive
}
}  // namespace

int rgrmhd_measure_fp64_peak(int device, int repeats, double* tflops_out) {
  if (!tflops_out || repeats < 1) return RGRMHD_E_INVALID;
  DeviceGuard guard(device);
  if (!guard.ok) return RGRMHD_E_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return RGRMHD_E_CUDA;
  double* out = nullptr;
  if (cudaMalloc((void**)&out, sizeof(double)) != cudaSuccess) return RGRMHD_E_NOMEM;
  cudaEvent_t a, b;
  if (cudaEventCreate(&a) != cudaSuccess) { cudaFree(out); return RGRMHD_E_CUDA; }
  if (cudaEventCreate(&b) != cudaSuccess) { cudaEventDestroy(a); cudaFree(out); return RGRMHD_E_CUDA; }
  const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 1 << 14;
  double best = 0.0;
  for (int r = 0; r < repeats + 1; ++r) {
    cudaEventRecord(a);
    k_dfma_peak<<<blocks, threads>>>(out, iters, 0.999999, 1e-9);
    cudaEventRecord(b);
    if (cudaEventSynchronize(b) != cudaSuccess) { cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(out); return RGRMHD_E_CUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    const double tf = 2.0 * 8.0 * (double)iters * blocks * threads / (ms * 1e-3) * 1e-12;
    if (r > 0 && tf > best) best = tf;   // first launch is warm-up
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  cudaFree(out);
  *tflops_out = best;
  return RGRMHD_OK;
}

int rgrmhd_launch_count(rgrmhd_t h, long long* host_out) {
  if (!h || !host_out) return RGRMHD_E_INVALID;
  *host_out = h->launches;
  return RGRMHD_OK;
}

const char* rgrmhd_strerror(int code) {
  switch (code) {
    case RGRMHD_OK: return "ok";
    case RGRMHD_E_INVALID: return "invalid argument";
    case RGRMHD_E_STATE: return "call out of order (metric / primitives / sigma not set, wrong sigma model, or a failed step left the state unusable until set_prims)";
    case RGRMHD_E_CUDA: return "CUDA error (see rgrmhd_last_cuda_error)";
    case RGRMHD_E_NOMEM: return "device allocation failed";
    case RGRMHD_E_TOO_LARGE: return "more cells than the fixed scratch array of rgrmhd_max_speed_static allows (RGRMHD_STATIC_MAX_CELLS)";
  }
  return "unknown status";
}

const char* rgrmhd_last_cuda_error(rgrmhd_t h) {
  return h ? h->last_error.c_str() : "";
}

}  // extern "C"
