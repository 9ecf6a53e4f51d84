// context.h -- the host-side context of libpycool.so, shared by the translation units of the library
// (pycool.cu: ABI and sequencing; models_*.cu: the kernel template instances of one model each).  Internal.
#pragma once
#include <cstdarg>
#include <cstdio>
#include <string>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/pycool.h"
#include "kernels.cuh"

namespace pycool {

constexpr int kMaxSumBlocks = 1184;      // capacity (partial sums) of the sum / energy kernels: 8 blocks per SM, at most
constexpr size_t kMaxSmem = 227 * 1024;  // dynamic shared memory one block may opt in to on sm_100
constexpr int kNumGeneric = 3;           // kick_fused variants (any N, any layout)
constexpr int kNumTiles = 13;            // + kick_tma variants (ghost layout only)

struct TileInfo { int tx, ty, nt, stages, xw; };   // stages > 0: TMA ring depth; xw: sites per thread along x (fp32)

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);


}  // namespace pycool

struct pycool_ctx {
  int N = 0, nf = 0, order = 0, model = 0, precision = 64;
  double L = 0, dx = 0, dt = 0, mpl = 1, rho_g = 0, rho_m = 0;
  size_t V = 0, elems = 0, esize = 8;
  double c[4] = {0, 0, 0, 0};
  pycool::ModelParams mp{};
  pycool::ScalarConst kc{};
  int nstages = 0;
  double w[16];
  // device memory: two state buffers (ping-pong), each phi and pi in layout L
  pycool::Layout lay{};
  void* phi[2] = {nullptr, nullptr};
  void* pi[2] = {nullptr, nullptr};
  int cur = 0;
  CUtensorMap tm[2][2];         // [buffer][phi, pi] for the current TMA tile
  double* partials = nullptr;   // max(3 * kick blocks, 13 * kMaxSumBlocks) doubles
  size_t partials_cap = 0;
  double* sums = nullptr;       // 16 doubles: reduced rows
  pycool_energy* d_energy = nullptr;   // the latest energy read-out, finished on the device (energy_finish)
  bool energy_through_drift = false;   // the next energy launch sees phi through the pending closing half drift
  // energy log (pycool_set_energy_cadence): every `log_every` completed steps an energy read-out is appended to a
  // device ring buffer by kernels enqueued from pycool_step, without a host synchronisation
  pycool_energy* d_log = nullptr;
  int log_every = 0, log_cap = 0;
  unsigned long long log_n = 0;        // entries written since the cadence was set
  unsigned long long steps_done = 0;   // completed steps since the cadence was set
  pycool::Scalars* sc = nullptr;
  unsigned int* ticket = nullptr;   // blocks-done counter of the fused stage tail (zero between launches)
  bool overlap_launch = true;       // kick_tma launched with programmatic stream serialization (PDL)
  int energy_tma = 1;               // pycool_energies through the TMA-fed kernel where the layout allows (0: plain;
                                    //   1: automatic variant; 2-4: a given variant, pycool_set_energy_kernel)
  int energy_nb = 0;                // blocks (= partial sums per quantity) of the latest energy launch
  bool persistent = true;           // kick_tma: one block per resident slot, the TMA ring runs on across items
  int blocks_launched = 0;          // grid size of the latest kick launch
  bool fused_tail = true;           // last block of a kick reduces the partials and advances the scalars
  bool cooperative = true;          // small lattices: several stages per cooperative launch (kick_tma_coop)
  int coop_ok = -1;                 // the device supports cooperative launches (-1: not asked yet)
  int coop_resident[16];            // co-resident blocks of kick_tma_coop per variant (-1: not asked yet, 0: not built)
  pycool::CoopSchedule coop{};      // schedule of the next cooperative launch
  pycool::StageLen len{};                   // stage weights handed to the next kick launch
  bool adaptive = false;            // dt is a physical-time increment (pycool_set_adaptive)
  int device = 0, sms = 0;          // the CUDA device this context lives on and its SM count
  int resident[16];                 // blocks of the kick variant that fit on the device at once (-1: not asked yet);
                                    //   asking also opts the instance in to its dynamic shared memory ON THIS DEVICE
  bool energy_attr[3] = {false, false, false};
  bool own_mem = false, own_stream = false;
  void* owned_block = nullptr;  // one allocation when own_mem
  cudaStream_t stream = nullptr;
  // launch geometry
  int tile = -1, zc = 0, zc_user = 0;
  dim3 grid;
  int region[2] = {1, 1};       // kick_tma item order: regions of region[0] x region[1] tiles (kick_tma.cuh: item_origin)
  int region_user = -1;         // pycool_set_item_order: -1 automatic, 0 plain x-y-z order, n > 0 about n tiles per region
  // state
  bool have_fields = false, nonfinite_seen = false;
  bool pending_drift = false;   // the closing half drift of the last step call is still to be applied to phi
  unsigned long long counts[4] = {0, 0, 0, 0};
  bool profiling = false;
  std::vector<cudaEvent_t> ev;   // pairs
  size_t ev_used = 0;
  double prof_ms = 0;
  unsigned long long prof_n = 0;
  std::string err;
};

namespace pycool {

// Record an error message in the context (or, without one, for pycool_last_error(NULL)) and return `code`.
int fail(pycool_ctx* c, int code, const char* fmt, ...);
#define CUDA_TRY(c, expr)                                                                                   \
  do {                                                                                                      \
    cudaError_t e_ = (expr);                                                                                \
    if (e_ != cudaSuccess) return ::pycool::fail((c), PYCOOL_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

// Every ABI entry runs on the context's device whatever device is current in the calling thread, and leaves the
// caller's current device as it found it (several contexts on several GPUs in one process: PAPER.md:511).
struct OnDevice {
  int prev = -1;
  explicit OnDevice(const pycool_ctx* c) {
    if (!c) return;
    int cur = -1;
    if (cudaGetDevice(&cur) == cudaSuccess && cur != c->device) {
      prev = cur;
      cudaSetDevice(c->device);
    }
  }
  ~OnDevice() { if (prev >= 0) cudaSetDevice(prev); }
  OnDevice(const OnDevice&) = delete;
  OnDevice& operator=(const OnDevice&) = delete;
};

extern const TileInfo kTiles[kNumTiles];

// Tensor map over one padded array: dims (x: N + 2 gx, y: N + 2 gy, z: N, f: nf), box (tx + 2 gx, ty + 2, 1, nf)
int encode_one(pycool_ctx* c, void* ptr, int tx, int ty, CUtensorMap* out);

// Kernel template instances live in one translation unit per model (models_*.cu); this is their one entry point.
enum Op { OP_KICK, OP_ENERGY, OP_SMEM, OP_RESIDENT, OP_BUILT, OP_KICK_COOP, OP_COOP_RESIDENT };
template <typename Real, class Model>
long long dispatch_one(pycool_ctx* c, Op op, int arg);

}  // namespace pycool
