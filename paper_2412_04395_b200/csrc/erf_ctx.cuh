// erf_ctx.cuh -- the context behind the opaque erf_ctx handle, and launch helpers.
#pragma once
#include <cuda_runtime.h>

#include <mutex>
#include <vector>

#include "../../include/erf_b200.h"
#include "erf_view.cuh"
#include "general_cells.cuh"

namespace erfb {

struct F5 {
  double *f[5];
};

// Kernel function attributes (the opt-in to more than 48 KB of dynamic shared memory) belong to a device's context, not
// to the process: a launch site keeps one OncePerDevice and sets its attributes the first time it runs on each GPU.
struct OncePerDevice {
  std::mutex mu;
  unsigned long long seen = 0;
  template <class F>
  void run(F set_attributes) {
    int dev = 0;
    const bool known = cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64;
    std::lock_guard<std::mutex> lock(mu);
    const unsigned long long bit = known ? 1ull << dev : 0;
    if (known && (seen & bit)) return;
    set_attributes();  // an unknown device index: every time (correct, only slower)
    seen |= bit;
  }
};

struct FusedState;  // fused.cuh

}  // namespace erfb

struct erf_ctx {
  int nx, ny, nz;
  size_t NW;  // elements of one 3-D array: nx*ny*(nz+1)
  erf_params p;
  erfb::View v;
  int path;
  int status;  // sticky error
  long long launches;
  long long bytes;
  std::vector<void *> allocs;

  // geometry (owned; v holds const aliases)
  double *zxf, *zyf, *zw, *hx, *hy, *hc, *zc, *hw, *hu, *hv, *sxw, *syw, *sxu, *syv;
  double *rho0, *Th0, *p0, *pi0;
  double *zl_dev;  // [(nz+1)] flat level heights (device) or null

  erfb::F5 S, St, R, P;  // S^n, stage state S^t, slow tendencies, perturbation S''
  double *theta_t, *pi_t;
  erfb::gen::Prim prim;  // general path intermediates
  double *Om_slow;      // contravariant flux of the stage state (general path)
  erfb::gen::Diff diff;
  bool diff_alloc;
  erfb::gen::Acou ac;
  erfb::FusedState *fz;  // fused flat-grid path (null until fused_setup)
  double *terr_U2, *terr_V2, *terr_rdzc;  // fused terrain substep kernel (k_acoustic_terrain.cu), allocated at first use

  // The terrain-general arrays (3-D metrics, base state, unfused intermediates) exist only where that path runs:
  // always on terrain / 3-D base states, on flat grids from the first use of ERF_PATH_GENERAL (ensure_general).
  bool gen_ready;
  double *base1d_r0, *base1d_T0;  // flat grid, 1-D base state: owned copies of the [nz] inputs (to build the 3-D arrays later)

  // one transported scalar (k_scalar.cu): rho*phi, its stage values, the sums of the substep momenta; null until
  // erf_set_scalar
  double *sc_Q, *sc_Qt, *sc_Qnew, *sc_sum[3], *sc_phi, *sc_R, *sc_G[2];

  // inflow boundaries [R:G30]: the Dirichlet column i = 0 ([5][nz+1][ny]) / row j = 0 ([5][nz+1][nx]) given to erf_set_state
  int inx, iny;
  double *in_x, *in_y;

  // anelastic mode (k_anelastic.cu): lagged p', the transform work arrays, twiddle and level tables; null until first use
  double *an_pp, *an_w[4], *an_tw, *an_lev;

  // ERF_OPT_GRAPH: one instantiated CUDA graph per buffer configuration of the fused step
  struct StepGraph {
    std::vector<const void *> before, after;  // buffer roles when the step starts / ends
    double dt;
    int ns;
    long long launches;
    long long last_use;  // graph_tick at the last launch (least recently used (dt, n_acoustic) pair goes first)
    cudaGraphExec_t exec;
  };
  bool graph_on, graph_warm;  // warm: a plain step has run (kernel attributes are set outside any capture)
  std::vector<StepGraph> graphs;
  long long graph_tick;

  // per-kernel timing (erf_set_timing)
  bool timing;
  struct TimedSpan { int id; cudaEvent_t a, b; };
  std::vector<TimedSpan> spans;
  std::vector<cudaEvent_t> event_pool;
  long long t_calls[ERF_TIMING_CLASSES];
  double t_ms[ERF_TIMING_CLASSES];

  double *alloc(size_t n);  // zero-initialised device doubles; null on failure (sets status)
};

namespace erfb {

// thread (i, j, k) from a 3-D launch: 32 x 8 threads over (x, y), one level per blockIdx.z (no index divisions)
template <class F>
__global__ void k_cells(int nx, int ny, int nlev, F f) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y, k = blockIdx.z;
  if (i >= nx || j >= ny || k >= nlev) return;
  f(i, j, k);
}

template <class F>
__global__ void k_columns(int nx, int ny, F f) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y;
  if (i >= nx || j >= ny) return;
  f(i, j);
}

template <class F>
inline void launch_cells(erf_ctx *c, cudaStream_t st, int nlev, F f) {
  if (nlev <= 0) return;
  dim3 block(32, 8), grid((c->nx + 31) / 32, (c->ny + 7) / 8, nlev);
  k_cells<<<grid, block, 0, st>>>(c->nx, c->ny, nlev, f);
  c->launches++;
}

template <class F>
inline void launch_columns(erf_ctx *c, cudaStream_t st, F f) {
  dim3 block(32, 4), grid((c->nx + 31) / 32, (c->ny + 3) / 4);
  k_columns<<<grid, block, 0, st>>>(c->nx, c->ny, f);
  c->launches++;
}

// Per-cell passes as functors over the view type: CTAs whose 32 x 8 tile lies at least MARGIN columns inside the domain
// run the body on a ViewNW (no wrap / clamp in the index helper), the others on the View.
constexpr int MARGIN = 3;

template <class F>
__global__ void __launch_bounds__(256) k_cells_v(View v, int nlev, F f) {
  // levels fastest in the launch order (vertical neighbours of the resident CTAs stay in L2)
  const int i = blockIdx.y * 32 + threadIdx.x, j = blockIdx.z * 8 + threadIdx.y, k = blockIdx.x;
  if (i >= v.nx || j >= v.ny || k >= nlev) return;
  const int x0 = blockIdx.y * 32, y0 = blockIdx.z * 8;
  const bool inner = x0 >= MARGIN && x0 + 32 + MARGIN <= v.nx && y0 >= MARGIN && y0 + 8 + MARGIN <= v.ny;
  if (inner) {
    const ViewNW vn(v);
    f(vn, i, j, k);
  } else {
    f(v, i, j, k);
  }
}

template <class F>
inline void launch_cells_v(erf_ctx *c, cudaStream_t st, int nlev, const F &f) {
  if (nlev <= 0) return;
  dim3 block(32, 8), grid(nlev, (c->nx + 31) / 32, (c->ny + 7) / 8);
  k_cells_v<<<grid, block, 0, st>>>(c->v, nlev, f);
  c->launches++;
}


}  // namespace erfb

namespace erfb {

// timing classes
enum { T_SLOW_GENERAL = 0, T_ACOUSTIC_GENERAL = 1, T_STAGE_GENERAL = 2, T_SLOW_FUSED = 3, T_VISC_FUSED = 4,
       T_ACOUSTIC_FUSED = 5, T_OTHER = 6 };

// brackets a region of launches on a stream with two events when timing is on
struct Timed {
  erf_ctx *c;
  cudaStream_t st;
  int idx;
  Timed(erf_ctx *c_, int id, cudaStream_t st_) : c(c_), st(st_), idx(-1) {
    if (!c->timing) return;
    erf_ctx::TimedSpan s;
    s.id = id;
    cudaEvent_t *ev[2] = {&s.a, &s.b};
    for (auto e : ev) {
      if (!c->event_pool.empty()) { *e = c->event_pool.back(); c->event_pool.pop_back(); }
      else if (cudaEventCreate(e) != cudaSuccess) return;
    }
    cudaEventRecord(s.a, st);
    c->spans.push_back(s);
    idx = (int)c->spans.size() - 1;
  }
  ~Timed() {
    if (idx >= 0) cudaEventRecord(c->spans[idx].b, st);
  }
};

// general path (k_general.cu).  ensure_general allocates and fills the 3-D metric / base-state arrays and the unfused
// intermediates on first use (returns the context status); every general_* function below requires it.
int ensure_general(erf_ctx *c, cudaStream_t st);
int build_general(erf_ctx *c, const gen::NodeH &Z, const double *rho0_in, const double *Th0_in, int base1d, cudaStream_t st);
bool ensure_prim(erf_ctx *c, bool all);  // u, v, w, p' (all: also theta, pi) work arrays
void impose_lids(erf_ctx *c, const F5 &S, cudaStream_t st);  // kinematic W on k = 0 and k = nz [R:G15]
// fills c->R, theta_t, pi_t; pan != null: the anelastic pressure-gradient / buoyancy pair with that p' (Sec. 2.2)
void general_slow_rhs(erf_ctx *c, const F5 &S, cudaStream_t st, const double *pan = nullptr);
void general_acoustic(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st);  // c->P in/out
void general_stage_init(erf_ctx *c, cudaStream_t st);    // P = S - St
void general_stage_finish(erf_ctx *c, cudaStream_t st);  // St += P, lids
void general_lids(erf_ctx *c, const F5 &S, cudaStream_t st);
void inflow_store(erf_ctx *c, cudaStream_t st);                  // remember column / row 0 of c->S
void inflow_impose(erf_ctx *c, const F5 &S, cudaStream_t st);    // write it back into S (every stage result)

// k_terrain_slow.cu: the advective tendencies of all five fields in one kernel (Eq. 17-21 stencils only)
bool terrain_advection_available(const erf_ctx *c);
void launch_terrain_advection(erf_ctx *c, const F5 &S, cudaStream_t st);

// k_anelastic.cu: RK2 + projection (Sec. 3.2 Eq. 14-16); flat, laterally periodic grids
int anelastic_step(erf_ctx *c, double dt, cudaStream_t st);
int anelastic_project(erf_ctx *c, const F5 &S, double dt, cudaStream_t st);

// k_scalar.cu: Eq. 4 after the substeps of a stage, with the time-averaged momenta (L138)
bool ensure_scalar(erf_ctx *c);
void scalar_stage(erf_ctx *c, const F5 &St, const double *Qt, const double *Qn, double *Qout, int nsub, double dts,
                  cudaStream_t st, bool folded = false);
void scalar_prepare_fused(erf_ctx *c, const F5 &St, const double *Qt, int nsub, cudaStream_t st);

// k_acoustic_terrain.cu: general_acoustic with the per-substep passes fused (terrain grids)
bool terrain_acoustic_available(const erf_ctx *c);
void terrain_acoustic(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st);

}  // namespace erfb
