// pycool.cu -- context, launch sequencing and the C ABI of libpycool.so (declared in include/pycool.h).
//
// The host side only validates arguments, owns buffers and enqueues kernels; a, p_a and every lattice sum live
// on the device, so pycool_step never synchronises (the paper copies the sums to the host at every sub-step,
// PAPER.md:395).  Sequence of one pycool_step(n) call, stages w_1..w_S (S = n * stages(order), h = w * step length):
//     scalar_update(mode 0, or 2 when the previous call's closing half drift is still pending)
//     for i in 1..S:  kick_tma / kick_fused: drift by c_drift, kick by h_i, sums; its last block reduces the
//                     partial sums and advances a, p_a, c_drift, kD, kV for stage i+1 (stage_finish)
//     (the closing half drift stays pending: the next call merges it, anything that reads phi applies it first)
// which is (2.48) composed per (2.43)-(2.45) with adjacent H1 and H2 halves merged.
// Other files: kick_tma.cuh (the hot kernel), kernels.cuh (scalars, generic kernel, pointwise kernels),
// energy_tma.cuh (pycool_energies), init_fields.cuh (initial conditions, spectra), potentials.cuh (models).
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <limits>
#include <new>
#include <string>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>
#include <dlfcn.h>

#include "context.h"
#include "cufft_api.h"
#include "init_fields.cuh"
#include "scalar_kernels.cuh"
#include "potentials.cuh"

using namespace pycool;

namespace {

// ---- stage weights: (2.42); (2.43)-(2.44) with n = 1 (reading G2); Table 1 ----
int stage_weights_ld(int order, long double* w) {
  if (order == 2) { w[0] = 1.0L; return 1; }
  if (order == 4) {
    const long double r = cbrtl(2.0L);
    w[0] = w[2] = 1.0L / (2.0L - r);
    w[1] = -r / (2.0L - r);
    return 3;
  }
  if (order == 6) {
    const long double t[3] = {0.78451361047755726382L, 0.23557321335935813368L, -1.17767998417887100695L};
    const long double mid = 1.0L - 2.0L * (t[0] + t[1] + t[2]);
    for (int i = 0; i < 3; ++i) w[i] = w[6 - i] = t[i];
    w[3] = mid;
    return 7;
  }
  if (order == 8) {
    const long double t[7] = {0.74167036435061295345L, -0.40910082580003159400L, 0.19075471029623837995L,
                              -0.57386247111608226666L, 0.29906418130365592384L, 0.33462491824529818378L,
                              0.31529309239676659663L};
    long double s = 0.0L;
    for (int i = 0; i < 7; ++i) { s += t[i]; w[i] = w[14 - i] = t[i]; }
    w[7] = 1.0L - 2.0L * s;
    return 15;
  }
  return 0;
}

thread_local std::string g_create_err = "no error";

}  // namespace

int pycool::fail(pycool_ctx* c, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (c) c->err = buf; else g_create_err = buf;
  return code;
}

//                                 generic kick_fused          | kick_tma (TX, TY, threads, ring stages)
const TileInfo pycool::kTiles[kNumTiles] = {{32, 8, 128, 0, 1}, {32, 16, 256, 0, 1}, {64, 8, 256, 0, 1},
                                            {64, 16, 256, 3, 2}, {32, 16, 128, 3, 2}, {128, 8, 256, 3, 2},
                                            {128, 16, 512, 3, 2}, {32, 16, 256, 3, 2}, {64, 8, 256, 3, 2},
                                            {128, 16, 256, 3, 2}, {32, 16, 256, 3, 2}, {128, 8, 256, 3, 4}, {32, 8, 128, 3, 2}};

namespace {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Ghost layout (TMA path) needs whole 16-byte pairs inside the lattice: N even.  Otherwise plain N^3.
Layout make_layout(int N, int nf, size_t esize) {
  Layout L{};
  L.N = N;
  if (N % 2 == 0 && N >= 4) {
    L.gx = (int)(16 / esize);
    L.gy = 1;
    L.pitch = (int)align_up((size_t)N + 2 * L.gx, 32 / esize);     // rows start on 32-byte sectors
    L.rows = N + 2;
  } else {
    L.gx = L.gy = 0;
    L.pitch = N;
    L.rows = N;
  }
  L.plane = (size_t)L.pitch * L.rows;
  L.field = L.plane * N;
  L.total = L.field * nf;
  return L;
}

// TMA variants need the ghost layout (even N); x quads need whole quads inside the lattice (N a multiple of 4)
bool tile_allowed(const Layout& L, int tile) {
  if (tile < kNumGeneric) return true;
  return L.gx > 0 && L.N % kTiles[tile].xw == 0;
}

int auto_tile(pycool_ctx* c);   // after dispatch(): needs the shared-memory size of a variant

int blocks_xy(int N, int tile) {
  const TileInfo& t = kTiles[tile];
  return ((N + t.tx - 1) / t.tx) * ((N + t.ty - 1) / t.ty);
}
int auto_zchunk(pycool_ctx* c);
// partial-sum capacity actually reserved: automatic geometry of every tile with zc >= min(N, 2)
size_t partials_capacity(int N) {
  size_t m = 13 * (size_t)kMaxSumBlocks;
  const int zmin = N < 2 ? N : 2;
  for (int t = 0; t < kNumTiles; ++t) {
    size_t b = 3 * (size_t)blocks_xy(N, t) * (size_t)((N + zmin - 1) / zmin);
    if (b > m) m = b;
  }
  return m;
}

// work memory: [phi0][pi0][phi1][pi1][partials][sums][scalars]
struct WorkLayout { size_t arr, off_part, off_sums, off_sc, total; };
WorkLayout work_layout(int N, int nf, size_t esize) {
  WorkLayout w;
  const Layout L = make_layout(N, nf, esize);
  w.arr = align_up(L.total * esize, 256);
  size_t o = 4 * w.arr;
  w.off_part = o; o += align_up(partials_capacity(N) * sizeof(double), 256);
  w.off_sums = o; o += 512;      // 16 reduced rows, then one pycool_energy (the latest read-out)
  w.off_sc = o; o += 256;
  w.total = o;
  return w;
}

bool valid_shape(int N, int nf, int precision) {
  return N >= 3 && N <= 2048 && nf >= 1 && nf <= 4 && (precision == 0 || precision == 32 || precision == 64);
}

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
    else
      cudaGetLastError();
  }
  return fn;
}

// Tensor map over one padded array: dims (x: N + 2 gx, y: N + 2 gy, z: N, f: nf), box (tx + 2 gx, ty + 2, 1, nf)
}  // namespace

int pycool::encode_one(pycool_ctx* c, void* ptr, int tx, int ty, CUtensorMap* out) {
  EncodeTiledFn enc = encode_fn();
  if (!enc) return fail(c, PYCOOL_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
  const Layout& L = c->lay;
  const cuuint64_t dims[4] = {(cuuint64_t)(L.N + 2 * L.gx), (cuuint64_t)(L.N + 2 * L.gy), (cuuint64_t)L.N,
                              (cuuint64_t)c->nf};
  const cuuint64_t strides[3] = {(cuuint64_t)L.pitch * c->esize, (cuuint64_t)L.plane * c->esize,
                                 (cuuint64_t)L.field * c->esize};
  const cuuint32_t box[4] = {(cuuint32_t)(tx + 2 * L.gx), (cuuint32_t)(ty + 2), 1u, (cuuint32_t)c->nf};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const CUtensorMapDataType dt = c->precision == 32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
  CUresult r = enc(out, dt, 4, ptr, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(c, PYCOOL_ECUDA, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
  return PYCOOL_OK;
}

namespace {

int encode_maps(pycool_ctx* c) {
  const TileInfo& t = kTiles[c->tile];
  for (int b = 0; b < 2; ++b)
    for (int a = 0; a < 2; ++a)
      if (int st = encode_one(c, a == 0 ? c->phi[b] : c->pi[b], t.tx, t.ty, &c->tm[b][a])) return st;
  return PYCOOL_OK;
}

// Kernel instances are compiled per model (models_*.cu, dispatch.cuh); here only the run-time selection.
template <typename Real>
long long dispatch_model(pycool_ctx* c, Op op, int arg) {
  switch (c->model) {
    case PYCOOL_FREE:
      switch (c->nf) {
        case 1: return dispatch_one<Real, Free<1>>(c, op, arg);
        case 2: return dispatch_one<Real, Free<2>>(c, op, arg);
        case 3: return dispatch_one<Real, Free<3>>(c, op, arg);
        default: return dispatch_one<Real, Free<4>>(c, op, arg);
      }
    case PYCOOL_CHAOTIC: return dispatch_one<Real, Chaotic>(c, op, arg);
    case PYCOOL_OSCILLON: return dispatch_one<Real, Oscillon>(c, op, arg);
    default: return dispatch_one<Real, QBall>(c, op, arg);
  }
}
long long dispatch(pycool_ctx* c, Op op, int arg) {
  return c->precision == 32 ? dispatch_model<float>(c, op, arg) : dispatch_model<double>(c, op, arg);
}

// Automatic variant (measured on B200, profiles/): the register-prefetch kernel where the layout has no ghosts
// (odd N); else the first TMA variant of a preference list whose ring fits in shared memory.
//   two fields fp64, one field fp32: 64 x 16 tile; two or more fields fp32: 128 x 8 (512-byte rows; the fp32
//   instances of both are cut for two blocks per SM, which is what fp32 needs: half the bytes per plane), as x quads
//   (variant 11: float4 accesses, 4 x 1 sites per thread; 2 % faster than the x pairs of variant 5 in one process at
//   512^3 and 1024^3, profiles/r2) when N is a multiple of 4;
//   one field fp64: 128 x 16 with 2 x 4 sites per thread (twice the work per plane and per barrier; a ring of 6
//   with the 64 x 16 tile gains nothing, so it is the per-plane fixed cost, not the bytes in flight);
//   Q-ball (bound by the latency of its dependent fp64 work): 32 x 8 with 2 x 1 sites per thread, four blocks per SM
//   (variant 12; 32 x 16 with two blocks per SM, variant 7, is 9 % slower in one process).
int auto_tile(pycool_ctx* c) {
  const Layout& L = c->lay;
  if (L.gx == 0) return L.N <= 64 ? 0 : 1;
  static const int pref_default[] = {3, 4}, pref_one[] = {9, 6, 3, 4}, pref_alu[] = {12, 7, 4}, pref_f32[] = {11, 5, 3, 4},
                   pref_small[] = {4, 10}, pref_many[] = {10, 4};
  const int* pref = pref_default;
  int n = 2;
  if (c->nf >= 3) { pref = c->precision == 64 ? pref_many : pref_small; n = 2; }   // 2 x 1 sites per thread in fp64
  else if (L.N <= 64) { pref = pref_small; n = 2; }
  else if (c->model == PYCOOL_QBALL && c->precision == 64) { pref = pref_alu; n = 3; }
  else if (c->nf == 1 && c->precision == 64) { pref = pref_one; n = 4; }
  else if (c->precision == 32 && c->nf >= 2) { pref = pref_f32; n = 4; }
  for (int i = 0; i < n; ++i)
    if (tile_allowed(L, pref[i]) && dispatch(c, OP_BUILT, pref[i])) return pref[i];
  return 1;
}

// Automatic z-chunk.  Every chunk marches two halo planes on top of its own (instructions and L2 traffic; since the
// region item order they are no longer DRAM traffic, kick_tma.cuh: item_origin), long chunks let x-y neighbours drift
// apart (their halo rows then miss L2) and leave fewer items to balance.  Measured inside sustained runs (bench.py,
// sw_power_cap, profiles/r2): fp64 64 x 16 tile at 512^3: 12 -> 0.903, 16 -> 0.920-0.924, 20 -> 0.931, 24 -> 0.927,
// 32 -> 0.902 of peak; at 1024^3: 16 -> 0.874, 24 -> 0.886, 32 -> 0.860; fp32 128 x 8 tile at 512^3: 16 -> 0.826,
// 24 -> 0.848, 32 -> 0.828; at 1024^3: 16 -> 0.794, 24 -> 0.809; its x-quad form (variant 11) is best at 32 planes.
// Small lattices: the chunk length that minimises
// rounds x (planes + 2 halo planes) + pipeline fill over the resident blocks.
int auto_zchunk(pycool_ctx* c) {
  const int N = c->N, bxy = blocks_xy(N, c->tile);
  if (N <= 16) return N;
  int R = (int)dispatch(c, OP_RESIDENT, c->tile);
  if (R < 1) R = c->sms;
  int cap = 16;
  if (c->precision == 64 && c->tile == 3) cap = N >= 1024 ? 24 : (N >= 512 ? 20 : 16);
  else if (c->precision == 32 && c->tile == 5) cap = N >= 512 ? 24 : 16;
  else if (c->precision == 32 && c->tile == 11) cap = N >= 512 ? 32 : 16;
  auto items = [&](int zc) { return (long long)bxy * ((N + zc - 1) / zc); };
  if (items(cap) >= 4LL * R) return cap;
  int best = cap < N ? cap : N;
  long long best_cost = -1;
  for (int zc = N; zc >= 1; --zc) {                           // small lattices: few planes per block; chunks are
    const int nbz = (N + zc - 1) / zc;                        // balanced, so what counts is the longest, ceil(N / nbz)
    const int len = (N + nbz - 1) / nbz;
    const long long rounds = ((long long)bxy * nbz + R - 1) / R;
    const long long cost = rounds * (len + 2) + 4;
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = len; }
  }
  return best;
}

int set_geometry(pycool_ctx* c) {
  const TileInfo& t = kTiles[c->tile];
  int zc = c->zc_user > 0 ? c->zc_user : auto_zchunk(c);
  if (zc > c->N) zc = c->N;
  // never exceed the reserved partial-sum capacity
  while (3 * (size_t)blocks_xy(c->N, c->tile) * (size_t)((c->N + zc - 1) / zc) > c->partials_cap) ++zc;
  c->zc = zc;
  c->grid = dim3((c->N + t.tx - 1) / t.tx, (c->N + t.ty - 1) / t.ty, (c->N + zc - 1) / zc);
  // item order (kick_tma.cuh: item_origin): regions of whole tile rows with about as many tiles as there are blocks
  // in flight (never more), the rows spread evenly over the regions; a layer that does not fit in flight even as a
  // single row, or a lattice whose whole x-y plane does, keeps the plain x-y-z order
  {
    const int nbx = (int)c->grid.x, nby = (int)c->grid.y;
    int ry = nby;
    if (t.stages > 0 && c->region_user != 0) {
      int R = (int)dispatch(c, OP_RESIDENT, c->tile);
      if (R < 1) R = c->sms;
      const int want = c->region_user > 0 ? c->region_user : R;
      const int ry_max = std::max(1, want / nbx);
      const int nreg = (nby + ry_max - 1) / ry_max;
      ry = (nby + nreg - 1) / nreg;
    }
    c->region[0] = nbx; c->region[1] = ry;
  }
  if (t.stages > 0) return encode_maps(c);
  return PYCOOL_OK;
}

int launch_scalar(pycool_ctx* c, const StageLen& len, int mode) {
  const int nb = (int)(c->grid.x * c->grid.y * c->grid.z);
  scalar_update<<<1, kReduceThreads, 0, c->stream>>>(c->sc, c->partials, nb, c->kc, len, mode);
  CUDA_TRY(c, cudaGetLastError());
  c->counts[1]++;
  return PYCOOL_OK;
}

int launch_flush(pycool_ctx* c) {
  const size_t n = c->lay.total;
  int nb = (int)std::min<size_t>((n + 255) / 256, (size_t)c->sms * 32);
  if (c->precision == 32)
    drift_flush<float><<<nb, 256, 0, c->stream>>>((float*)c->phi[c->cur], (const float*)c->pi[c->cur], c->sc, n);
  else
    drift_flush<double><<<nb, 256, 0, c->stream>>>((double*)c->phi[c->cur], (const double*)c->pi[c->cur], c->sc, n);
  CUDA_TRY(c, cudaGetLastError());
  c->counts[2]++;
  return PYCOOL_OK;
}

// The closing half drift of a pycool_step call is deferred: a following pycool_step merges it with its own
// opening half drift (exactly as between two stages of one call, so step(1) x n == step(n) bit for bit); anything
// that looks at phi applies it first.
int ensure_flushed(pycool_ctx* c) {
  if (!c->pending_drift) return PYCOOL_OK;
  c->pending_drift = false;
  return launch_flush(c);
}

int launch_sum_pi2(pycool_ctx* c) {
  const size_t n = c->elems;
  int nb = (int)std::min<size_t>((n + 255) / 256, (size_t)kMaxSumBlocks);
  if (c->precision == 32) sumsq<float><<<nb, 256, 0, c->stream>>>((const float*)c->pi[c->cur], c->lay, c->nf, c->partials);
  else sumsq<double><<<nb, 256, 0, c->stream>>>((const double*)c->pi[c->cur], c->lay, c->nf, c->partials);
  CUDA_TRY(c, cudaGetLastError());
  reduce_rows<<<1, kReduceThreads, 0, c->stream>>>(c->partials, nb, c->sums);
  CUDA_TRY(c, cudaGetLastError());
  store_spi2<<<1, 1, 0, c->stream>>>(c->sc, c->sums);
  CUDA_TRY(c, cudaGetLastError());
  c->counts[3] += 3;
  return PYCOOL_OK;
}

// Copy between a dense [nf][N][N][N] array (host or device) and a state array in layout L.
int copy_dense(pycool_ctx* c, void* state, void* dense, bool to_state, cudaMemcpyKind kind) {
  const Layout& L = c->lay;
  cudaMemcpy3DParms p;
  std::memset(&p, 0, sizeof p);
  const cudaPitchedPtr ps = make_cudaPitchedPtr(state, (size_t)L.pitch * c->esize, (size_t)L.pitch, (size_t)L.rows);
  const cudaPitchedPtr pd = make_cudaPitchedPtr(dense, (size_t)L.N * c->esize, (size_t)L.N, (size_t)L.N);
  const cudaPos pos_s = make_cudaPos((size_t)L.gx * c->esize, (size_t)L.gy, 0), pos_d = make_cudaPos(0, 0, 0);
  if (to_state) { p.srcPtr = pd; p.srcPos = pos_d; p.dstPtr = ps; p.dstPos = pos_s; }
  else { p.srcPtr = ps; p.srcPos = pos_s; p.dstPtr = pd; p.dstPos = pos_d; }
  p.extent = make_cudaExtent((size_t)L.N * c->esize, (size_t)L.N, (size_t)L.N * c->nf);
  p.kind = kind;
  CUDA_TRY(c, cudaMemcpy3DAsync(&p, c->stream));
  return PYCOOL_OK;
}

int launch_fill_ghosts(pycool_ctx* c, void* arr) {
  const Layout& L = c->lay;
  if (L.gx == 0) return PYCOOL_OK;
  const size_t n = (size_t)(L.N + 2 * L.gx) * (L.N + 2 * L.gy) * L.N * c->nf;
  const int nb = (int)std::min<size_t>((n + 255) / 256, (size_t)c->sms * 32);
  if (c->precision == 32) fill_ghosts<float><<<nb, 256, 0, c->stream>>>((float*)arr, L, c->nf);
  else fill_ghosts<double><<<nb, 256, 0, c->stream>>>((double*)arr, L, c->nf);
  CUDA_TRY(c, cudaGetLastError());
  c->counts[3]++;
  return PYCOOL_OK;
}

// One energy read-out, kernels only (no host synchronisation): the lattice sums of the current buffers -- seen through
// the pending closing half drift when `through_drift` -- then energy_finish into *d_out (device).
int enqueue_energy(pycool_ctx* c, bool through_drift, pycool_energy* d_out) {
  int nb = (int)std::min<size_t>((c->V + 255) / 256, (size_t)kMaxSumBlocks);
  c->energy_through_drift = through_drift;
  int st = (int)dispatch(c, OP_ENERGY, nb);
  c->energy_through_drift = false;
  if (st != PYCOOL_OK) return st;
  EnergyConst k;
  k.V = (double)c->V; k.dx2 = c->dx * c->dx; k.mpl = c->mpl; k.rho_g = c->rho_g; k.rho_m = c->rho_m; k.nf = c->nf;
  energy_finish<<<1, kReduceThreads, 0, c->stream>>>(c->partials, c->energy_nb, c->sc, k, d_out);
  CUDA_TRY(c, cudaGetLastError());
  c->counts[3] += 2;
  return PYCOOL_OK;
}

int read_scalars(pycool_ctx* c, Scalars* s) {
  CUDA_TRY(c, cudaMemcpyAsync(s, c->sc, sizeof(Scalars), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (s->nonfinite) {
    c->nonfinite_seen = true;
    return fail(c, PYCOOL_ENONFINITE, "a lattice sum became non-finite");
  }
  return PYCOOL_OK;
}

// The energies of the time-synchronised state on the host: flush, read-out on the device, one D2H copy; synchronises.
int energies_now(pycool_ctx* c, pycool_energy* o) {
  int st = ensure_flushed(c);
  if (st == PYCOOL_OK) st = enqueue_energy(c, false, c->d_energy);
  if (st != PYCOOL_OK) return st;
  CUDA_TRY(c, cudaMemcpyAsync(o, c->d_energy, sizeof(pycool_energy), cudaMemcpyDeviceToHost, c->stream));
  Scalars s;
  return read_scalars(c, &s);
}

// ---- cuFFT, loaded on first use (cufft_api.h)
}  // namespace
const CufftApi& pycool::cufft_api() {
  static CufftApi api;
  static bool tried = false;
  if (tried) return api;
  tried = true;
  void* h = nullptr;
  for (const char* name : {"libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so.11"}) {
    h = dlopen(name, RTLD_NOW | RTLD_LOCAL);
    if (h) break;
  }
  if (!h) return api;
  api.plan3d = (decltype(api.plan3d))dlsym(h, "cufftPlan3d");
  api.set_stream = (decltype(api.set_stream))dlsym(h, "cufftSetStream");
  api.exec_z2d = (decltype(api.exec_z2d))dlsym(h, "cufftExecZ2D");
  api.exec_d2z = (decltype(api.exec_d2z))dlsym(h, "cufftExecD2Z");
  api.destroy = (decltype(api.destroy))dlsym(h, "cufftDestroy");
  api.ok = api.plan3d && api.set_stream && api.exec_z2d && api.exec_d2z && api.destroy;
  return api;
}
namespace {

template <typename Real>
int init_one_array(pycool_ctx* c, const CufftApi& fft, cufftHandle plan, double2* scratch, Real* dst,
                   const Spectrum& sp, uint32_t aid, unsigned long long seed) {
  const int N = c->N;
  const size_t nmodes = (size_t)N * N * (N / 2 + 1);
  int nb = (int)std::min<size_t>((nmodes + 255) / 256, (size_t)c->sms * 64);
  fill_spectrum<<<nb, 256, 0, c->stream>>>(scratch, N, c->L, sp, aid, seed);
  CUDA_TRY(c, cudaGetLastError());
  if (fft.exec_z2d(plan, (cufftDoubleComplex*)scratch, (cufftDoubleReal*)scratch) != CUFFT_SUCCESS)
    return fail(c, PYCOOL_ECUDA, "cufftExecZ2D failed");
  nb = (int)std::min<size_t>((c->V + 255) / 256, (size_t)c->sms * 64);
  const double scale = std::sqrt(2.0) / (c->L * std::sqrt(c->L));
  scatter_real<Real><<<nb, 256, 0, c->stream>>>(dst, c->lay, (const double*)scratch, sp.mean, scale);
  CUDA_TRY(c, cudaGetLastError());
  c->counts[3] += 2;
  return PYCOOL_OK;
}

int create_common(pycool_ctx** out, int N, double L, int nf, const pycool_params* p, int order, double dt,
                  void* d_work, size_t work_bytes, void* stream, bool ext) {
  if (!out) return fail(nullptr, PYCOOL_EINVAL, "out is NULL");
  *out = nullptr;
  if (!p) return fail(nullptr, PYCOOL_EINVAL, "params is NULL");
  if (!valid_shape(N, nf, p->precision)) return fail(nullptr, PYCOOL_EINVAL, "N must be 3..2048, nfields 1..4, precision 0/32/64");
  if (!(L > 0) || !std::isfinite(L)) return fail(nullptr, PYCOOL_EINVAL, "L must be finite and > 0");
  long double wl[16];
  const int ns = stage_weights_ld(order, wl);
  if (ns == 0) return fail(nullptr, PYCOOL_EINVAL, "order must be 2, 4, 6 or 8");
  if (dt == 0 || !std::isfinite(dt)) return fail(nullptr, PYCOOL_EINVAL, "dt must be finite and non-zero");
  if (p->model < PYCOOL_FREE || p->model > PYCOOL_QBALL) return fail(nullptr, PYCOOL_EINVAL, "unknown model");
  if ((p->model == PYCOOL_CHAOTIC || p->model == PYCOOL_QBALL) && nf != 2)
    return fail(nullptr, PYCOOL_EINVAL, "this model needs nfields = 2");
  if (p->model == PYCOOL_OSCILLON && nf != 1) return fail(nullptr, PYCOOL_EINVAL, "oscillon needs nfields = 1");
  if (!(p->mpl > 0)) return fail(nullptr, PYCOOL_EINVAL, "mpl must be > 0 (+INF = static background)");
  if (p->model == PYCOOL_QBALL && !(p->p[2] > 0)) return fail(nullptr, PYCOOL_EINVAL, "Q-ball needs M^2 > 0");
  const double* cs = p->stencil;
  const bool dflt = cs[0] == 0 && cs[1] == 0 && cs[2] == 0 && cs[3] == 0;
  if (!dflt) {
    const double s = 6 * cs[1] + 12 * cs[2] + 8 * cs[3];
    if (!(std::fabs(cs[0] + s) <= 1e-12 * (std::fabs(cs[0]) + std::fabs(s))))
      return fail(nullptr, PYCOOL_EINVAL, "stencil must satisfy c0 = -(6 c1 + 12 c2 + 8 c3)");
  }
  if (ext && !d_work) return fail(nullptr, PYCOOL_EINVAL, "work buffer is NULL");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(nullptr, PYCOOL_ECUDA, "no CUDA device: libpycool has no CPU path");
  }
  pycool_ctx* c = new (std::nothrow) pycool_ctx();
  if (!c) return fail(nullptr, PYCOOL_ENOMEM, "host allocation failed");
  for (int& r : c->resident) r = -1;
  for (int& r : c->coop_resident) r = -1;
  {
    // the context lives on the device of the caller's work buffer (ext), else on the current device
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && ext) {
      cudaPointerAttributes pa;
      e = cudaPointerGetAttributes(&pa, d_work);
      if (e == cudaSuccess && pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) {
        delete c;
        return fail(nullptr, PYCOOL_EINVAL, "work buffer is not device memory");
      }
      if (e == cudaSuccess) dev = pa.device;
    }
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess || c->sms < 1) {
      cudaGetLastError();
      delete c;
      return fail(nullptr, PYCOOL_ECUDA, "cannot query the CUDA device: %s", cudaGetErrorString(e));
    }
    c->device = dev;
  }
  OnDevice on_device(c);
  c->N = N; c->nf = nf; c->order = order; c->model = p->model;
  c->precision = p->precision == 32 ? 32 : 64;
  c->esize = c->precision == 32 ? 4 : 8;
  c->L = L; c->dx = L / N; c->dt = dt; c->mpl = p->mpl; c->rho_g = p->rho_gamma0; c->rho_m = p->rho_m0;
  c->V = (size_t)N * N * N; c->elems = c->V * nf;
  c->lay = make_layout(N, nf, c->esize);
  if (dflt) { c->c[0] = -128.0 / 30.0; c->c[1] = 14.0 / 30.0; c->c[2] = 3.0 / 30.0; c->c[3] = 1.0 / 30.0; }
  else for (int i = 0; i < 4; ++i) c->c[i] = cs[i];
  for (int i = 0; i < 8; ++i) c->mp.p[i] = p->p[i];
  c->mp.inv_mpl2 = std::isinf(p->mpl) ? 0.0 : 1.0 / (p->mpl * p->mpl);
  c->kc.den = 6.0 * (double)c->V * p->mpl * p->mpl;
  c->kc.Vrho_m = (double)c->V * p->rho_m0;
  c->kc.dx2 = c->dx * c->dx;
  c->nstages = ns;
  for (int i = 0; i < ns; ++i) c->w[i] = (double)wl[i];

  const WorkLayout w = work_layout(N, nf, c->esize);
  unsigned char* work = nullptr;
  int rc = PYCOOL_OK;
  if (ext) {
    if (work_bytes < w.total) { rc = fail(nullptr, PYCOOL_EINVAL, "work buffer too small: need %zu bytes", w.total); goto bad; }
    if (((uintptr_t)d_work & 255) != 0) { rc = fail(nullptr, PYCOOL_EINVAL, "work buffer must be 256-byte aligned"); goto bad; }
    work = (unsigned char*)d_work;
    c->stream = (cudaStream_t)stream;
  } else {
    void* blk = nullptr;
    if (cudaMalloc(&blk, w.total) != cudaSuccess) {
      cudaGetLastError();
      rc = fail(nullptr, PYCOOL_ENOMEM, "cudaMalloc of %zu bytes failed", w.total);
      goto bad;
    }
    c->owned_block = blk; c->own_mem = true;
    work = (unsigned char*)blk;
    if (cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) != cudaSuccess) {
      cudaGetLastError();
      rc = fail(nullptr, PYCOOL_ECUDA, "cudaStreamCreate failed");
      goto bad;
    }
    c->own_stream = true;
  }
  c->phi[0] = work; c->pi[0] = work + w.arr;
  c->phi[1] = work + 2 * w.arr; c->pi[1] = work + 3 * w.arr;
  c->partials = (double*)(work + w.off_part);
  c->partials_cap = partials_capacity(N);
  c->sums = (double*)(work + w.off_sums);
  c->d_energy = (pycool_energy*)(work + w.off_sums + 256);
  c->sc = (Scalars*)(work + w.off_sc);
  c->ticket = (unsigned int*)(work + w.off_sc + 128);
  c->tile = auto_tile(c);
  {
    // padding and ghosts start as zeros (the closing drift sweeps the whole padded arrays)
    Scalars s0;
    std::memset(&s0, 0, sizeof s0);
    s0.a = 1.0; s0.a_sync = 1.0;
    if (cudaMemsetAsync(work, 0, 4 * w.arr, c->stream) != cudaSuccess ||
        cudaMemsetAsync(work + w.off_sc, 0, 256, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(c->sc, &s0, sizeof s0, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess) {
      rc = fail(nullptr, PYCOOL_ECUDA, "initialising device memory failed: %s", cudaGetErrorString(cudaGetLastError()));
      goto bad;
    }
  }
  rc = set_geometry(c);
  if (rc != PYCOOL_OK) { g_create_err = c->err; goto bad; }
  *out = c;
  return PYCOOL_OK;
bad:
  if (c->own_stream) cudaStreamDestroy(c->stream);
  if (c->owned_block) cudaFree(c->owned_block);
  delete c;
  return rc;
}

}  // namespace

// =================================================================================================== C ABI
extern "C" {

int pycool_create(pycool_ctx** out, int N, double L, int nfields, const pycool_params* params, int order,
                  double dt) {
  return create_common(out, N, L, nfields, params, order, dt, nullptr, 0, nullptr, false);
}

size_t pycool_work_bytes(int N, int nfields, int precision) {
  if (!valid_shape(N, nfields, precision)) return 0;
  return work_layout(N, nfields, precision == 32 ? 4 : 8).total;
}

int pycool_create_ext(pycool_ctx** out, int N, double L, int nfields, const pycool_params* params, int order,
                      double dt, void* d_work, size_t work_bytes, void* cuda_stream) {
  return create_common(out, N, L, nfields, params, order, dt, d_work, work_bytes, cuda_stream, true);
}

static int upload(pycool_ctx* c, const void* phi, const void* pi, cudaMemcpyKind kind) {
  c->cur = 0;
  c->pending_drift = false;
  int st = copy_dense(c, c->phi[0], const_cast<void*>(phi), true, kind);
  if (st == PYCOOL_OK) st = copy_dense(c, c->pi[0], const_cast<void*>(pi), true, kind);
  if (st == PYCOOL_OK) st = launch_fill_ghosts(c, c->phi[0]);
  if (st == PYCOOL_OK) st = launch_fill_ghosts(c, c->pi[0]);
  if (st != PYCOOL_OK) return st;
  c->have_fields = true;
  c->nonfinite_seen = false;
  CUDA_TRY(c, cudaMemsetAsync(&c->sc->nonfinite, 0, sizeof(int), c->stream));
  return launch_sum_pi2(c);
}

int pycool_set_fields(pycool_ctx* c, const void* phi_host, const void* pi_host) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!phi_host || !pi_host) return fail(c, PYCOOL_EINVAL, "phi_host / pi_host is NULL");
  int st = upload(c, phi_host, pi_host, cudaMemcpyHostToDevice);
  if (st != PYCOOL_OK) return st;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return PYCOOL_OK;
}

int pycool_set_fields_device(pycool_ctx* c, const void* d_phi_src, const void* d_pi_src) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!d_phi_src || !d_pi_src) return fail(c, PYCOOL_EINVAL, "source pointer is NULL");
  return upload(c, d_phi_src, d_pi_src, cudaMemcpyDeviceToDevice);
}

int pycool_init_fields(pycool_ctx* c, unsigned long long seed, const pycool_spectrum* phi_spec,
                       const pycool_spectrum* pi_spec) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!phi_spec || !pi_spec) return fail(c, PYCOOL_EINVAL, "phi_spec / pi_spec is NULL");
  if (c->N % 2) return fail(c, PYCOOL_EINVAL, "pycool_init_fields needs an even N (Hermitian planes ix = 0, N/2)");
  for (int f = 0; f < c->nf; ++f)
    for (const pycool_spectrum* sp : {phi_spec + f, pi_spec + f})
      if (!std::isfinite(sp->mean) || !std::isfinite(sp->amp) || !std::isfinite(sp->m2) || !std::isfinite(sp->q) ||
          !std::isfinite(sp->kmax) || sp->m2 < 0)
        return fail(c, PYCOOL_EINVAL, "spectrum parameters must be finite, m2 >= 0");
  const CufftApi& fft = cufft_api();
  if (!fft.ok) return fail(c, PYCOOL_ECUDA, "cuFFT (libcufft.so.11) could not be loaded");
  const int N = c->N;
  double2* scratch = nullptr;
  CUDA_TRY(c, cudaMalloc(&scratch, (size_t)N * N * (N / 2 + 1) * sizeof(double2)));
  cufftHandle plan = 0;
  int st = PYCOOL_OK;
  if (fft.plan3d(&plan, N, N, N, CUFFT_Z2D) != CUFFT_SUCCESS || fft.set_stream(plan, c->stream) != CUFFT_SUCCESS) {
    cudaFree(scratch);
    return fail(c, PYCOOL_ENOMEM, "cufftPlan3d(%d^3, Z2D) failed", N);
  }
  c->cur = 0;
  c->pending_drift = false;
  for (int f = 0; f < c->nf && st == PYCOOL_OK; ++f)
    for (int kind = 0; kind < 2 && st == PYCOOL_OK; ++kind) {
      const pycool_spectrum& u = kind == 0 ? phi_spec[f] : pi_spec[f];
      const Spectrum sp{u.mean, u.amp, u.m2, u.q, u.kmax};
      void* base = kind == 0 ? c->phi[0] : c->pi[0];
      if (c->precision == 32)
        st = init_one_array<float>(c, fft, plan, scratch, (float*)base + (size_t)f * c->lay.field, sp, 2u * f + kind, seed);
      else
        st = init_one_array<double>(c, fft, plan, scratch, (double*)base + (size_t)f * c->lay.field, sp, 2u * f + kind, seed);
    }
  cudaError_t e = cudaStreamSynchronize(c->stream);
  fft.destroy(plan);
  cudaFree(scratch);
  if (st != PYCOOL_OK) return st;
  CUDA_TRY(c, e);
  c->have_fields = true;
  c->nonfinite_seen = false;
  CUDA_TRY(c, cudaMemsetAsync(&c->sc->nonfinite, 0, sizeof(int), c->stream));
  return launch_sum_pi2(c);
}

namespace {

// D2Z transform of one array of the current state (phi or pi of one field) into `scratch` (N^2 (N/2+1) complex).
int transform_array(pycool_ctx* c, const CufftApi& fft, cufftHandle plan, int field, int which, double2* scratch) {
  const int nb = (int)std::min<size_t>((c->V + 255) / 256, (size_t)c->sms * 64);
  const void* base = which == 0 ? c->phi[c->cur] : c->pi[c->cur];
  if (c->precision == 32)
    gather_real<float><<<nb, 256, 0, c->stream>>>((double*)scratch, (const float*)base + (size_t)field * c->lay.field, c->lay);
  else
    gather_real<double><<<nb, 256, 0, c->stream>>>((double*)scratch, (const double*)base + (size_t)field * c->lay.field, c->lay);
  CUDA_TRY(c, cudaGetLastError());
  c->counts[3]++;
  if (fft.exec_d2z(plan, (cufftDoubleReal*)scratch, (cufftDoubleComplex*)scratch) != CUFFT_SUCCESS)
    return fail(c, PYCOOL_ECUDA, "cufftExecD2Z failed");
  return PYCOOL_OK;
}

// Shell sums of one (kind 0: |F|^2 of one array; kind 1: number and energy density of one field) spectrum.
int shell_spectrum(pycool_ctx* c, int field, int which, int kind, double m_eff2, int nbins, double* out0, double* out1,
                   double* count_host) {
  const CufftApi& fft = cufft_api();
  if (!fft.ok) return fail(c, PYCOOL_ECUDA, "cuFFT (libcufft.so.11) could not be loaded");
  const int N = c->N, rows = kind == 0 ? 2 : 3;
  const size_t nmodes = (size_t)N * N * (N / 2 + 1);
  const int nblk = (int)std::min<size_t>((nmodes + 255) / 256, (size_t)c->sms * 8);
  Scalars sc;
  int st = read_scalars(c, &sc);                           // the time-synchronised a (the state has been flushed)
  if (st != PYCOOL_OK) return st;
  double2* scratch = nullptr;
  double* part = nullptr;
  if (cudaMalloc(&scratch, (kind == 0 ? 1 : 2) * nmodes * sizeof(double2)) != cudaSuccess ||
      cudaMalloc(&part, ((size_t)nblk + 1) * rows * nbins * sizeof(double)) != cudaSuccess) {
    cudaGetLastError();
    if (scratch) cudaFree(scratch);
    return fail(c, PYCOOL_ENOMEM, "out of device memory for the spectrum scratch");
  }
  cufftHandle plan = 0;
  if (fft.plan3d(&plan, N, N, N, CUFFT_D2Z) != CUFFT_SUCCESS || fft.set_stream(plan, c->stream) != CUFFT_SUCCESS) {
    cudaFree(scratch); cudaFree(part);
    return fail(c, PYCOOL_ENOMEM, "cufftPlan3d(%d^3, D2Z) failed", N);
  }
  const double norm = c->L * std::sqrt(c->L) / (std::sqrt(2.0) * (double)N * (double)N * (double)N);
  std::vector<double> h((size_t)rows * nbins);
  auto run = [&]() -> int {
    if (kind == 0) {
      if (int e = transform_array(c, fft, plan, field, which, scratch)) return e;
      bin_shells<<<nblk, 256, 2 * nbins * sizeof(double), c->stream>>>(scratch, N, norm * norm, nbins, part);
    } else {
      if (int e = transform_array(c, fft, plan, field, 0, scratch)) return e;
      if (int e = transform_array(c, fft, plan, field, 1, scratch + nmodes)) return e;
      ModeSpectrumArgs g;
      g.norm2 = norm * norm; g.a2 = sc.a_sync * sc.a_sync; g.m_eff2 = m_eff2; g.inv_dx2 = 1.0 / (c->dx * c->dx);
      g.c0 = c->c[0]; g.c1 = c->c[1]; g.c2 = c->c[2]; g.c3 = c->c[3];
      bin_mode_spectra<<<nblk, 256, 3 * nbins * sizeof(double), c->stream>>>(scratch, scratch + nmodes, N, g, nbins, part);
    }
    CUDA_TRY(c, cudaGetLastError());
    double* out = part + (size_t)nblk * rows * nbins;
    reduce_shells<<<(rows * nbins + 255) / 256, 256, 0, c->stream>>>(part, nblk, rows * nbins, out);
    CUDA_TRY(c, cudaGetLastError());
    c->counts[3] += 2;
    CUDA_TRY(c, cudaMemcpyAsync(h.data(), out, h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return PYCOOL_OK;
  };
  st = run();
  if (st != PYCOOL_OK) cudaStreamSynchronize(c->stream);
  fft.destroy(plan);
  cudaFree(scratch); cudaFree(part);
  if (st != PYCOOL_OK) return st;
  for (int i = 0; i < nbins; ++i) {
    out0[i] = h[i];
    if (kind != 0) out1[i] = h[nbins + i];
    count_host[i] = h[(size_t)(rows - 1) * nbins + i];
  }
  return PYCOOL_OK;
}

}  // namespace

int pycool_field_spectrum(pycool_ctx* c, int field, int which, int nbins, double* power_host, double* count_host) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!c->have_fields) return fail(c, PYCOOL_ESTATE, "spectrum before set_fields");
  if (field < 0 || field >= c->nf || (which != 0 && which != 1)) return fail(c, PYCOOL_EINVAL, "bad field / which");
  if (nbins < 1 || nbins > 3072 || !power_host || !count_host)   // 2 nbins doubles of shared memory, <= 48 KB
    return fail(c, PYCOOL_EINVAL, "nbins must be 1..3072 and the outputs non-NULL");
  int st = ensure_flushed(c);
  if (st != PYCOOL_OK) return st;
  return shell_spectrum(c, field, which, 0, 0.0, nbins, power_host, nullptr, count_host);
}

int pycool_mode_spectra(pycool_ctx* c, int field, double m_eff2, int nbins, double* number_host, double* energy_host,
                        double* count_host) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!c->have_fields) return fail(c, PYCOOL_ESTATE, "spectrum before set_fields");
  if (field < 0 || field >= c->nf || !std::isfinite(m_eff2)) return fail(c, PYCOOL_EINVAL, "bad field or m_eff2");
  if (nbins < 1 || nbins > 2048 || !number_host || !energy_host || !count_host)   // 3 nbins doubles of shared memory
    return fail(c, PYCOOL_EINVAL, "nbins must be 1..2048 and the outputs non-NULL");
  int st = ensure_flushed(c);
  if (st != PYCOOL_OK) return st;
  return shell_spectrum(c, field, 0, 1, m_eff2, nbins, number_host, energy_host, count_host);
}

int pycool_set_background(pycool_ctx* c, double a, double p_a) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!(a > 0) || !std::isfinite(a)) return fail(c, PYCOOL_EINVAL, "a must be finite and > 0");
  if (int st = ensure_flushed(c)) return st;
  if (std::isnan(p_a)) {                                   // reading G10: (2.18), expanding branch
    if (!c->have_fields) return fail(c, PYCOOL_ESTATE, "p_a = NaN needs fields (call set_fields first)");
    if (std::isinf(c->mpl)) return fail(c, PYCOOL_EINVAL, "p_a = NaN with a static background (mpl = INF)");
    set_scalars<<<1, 1, 0, c->stream>>>(c->sc, a, 0.0, 0);   // rho at the new a
    CUDA_TRY(c, cudaGetLastError());
    pycool_energy e;
    int st = energies_now(c, &e);
    if (st != PYCOOL_OK) return st;
    if (!(e.rho >= 0)) return fail(c, PYCOOL_EINVAL, "negative or non-finite energy density");
    const double ap = a * a * (double)sqrtl((long double)(e.rho / 3.0)) / c->mpl;   // (2.18)
    p_a = -6.0 * (double)c->V * c->mpl * c->mpl * ap;                                // (2.11)
  }
  set_scalars<<<1, 1, 0, c->stream>>>(c->sc, a, p_a, 1);
  CUDA_TRY(c, cudaGetLastError());
  return PYCOOL_OK;
}

int pycool_set_dt(pycool_ctx* c, double dt) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (dt == 0 || !std::isfinite(dt)) return fail(c, PYCOOL_EINVAL, "dt must be finite and non-zero");
  c->dt = dt;
  return PYCOOL_OK;
}

int pycool_step(pycool_ctx* c, int nsteps) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!c->have_fields) return fail(c, PYCOOL_ESTATE, "step before set_fields");
  if (nsteps < 0) return fail(c, PYCOOL_EINVAL, "nsteps < 0");
  if (c->nonfinite_seen) return fail(c, PYCOOL_ENONFINITE, "a lattice sum became non-finite");
  if (nsteps == 0) return PYCOOL_OK;
  const int ns = c->nstages;
  const long long S = (long long)nsteps * ns;
  StageLen len;
  len.dt = c->dt;
  len.adaptive = c->adaptive ? 1 : 0;
  len.w = 0.0; len.w_next = c->w[0]; len.ends_step = 0;
  int st = launch_scalar(c, len, c->pending_drift ? 2 : 0);
  if (st != PYCOOL_OK) return st;
  if (c->profiling && c->ev.size() < c->ev_used + 2 * (size_t)S) {
    const size_t want = c->ev_used + 2 * (size_t)S;
    while (c->ev.size() < want) {
      cudaEvent_t e;
      CUDA_TRY(c, cudaEventCreate(&e));
      c->ev.push_back(e);
    }
  }
  // Small lattices whose work items are all co-resident: several stages per cooperative launch, a grid barrier
  // between stages instead of a kernel boundary (kick_tma.cuh: kick_tma_coop); same results bit for bit.
  const long long nitems = (long long)c->grid.x * c->grid.y * c->grid.z;
  bool coop = c->cooperative && c->fused_tail && !c->profiling && kTiles[c->tile].stages > 0 &&
                    dispatch(c, OP_COOP_RESIDENT, c->tile) >= nitems &&
                    6 * nitems <= (long long)c->partials_cap;   // two sets of partial sums, by stage parity
  for (long long i = 0; i < S;) {
    if (coop) {
      // up to the end of the call, the next energy-log point, or 32 steps, whichever comes first
      long long n = std::min<long long>(S - i, 32LL * ns);
      if (c->log_every > 0) {
        const long long to_step_end = ns - (i % ns);
        const unsigned long long steps_to_log = (unsigned long long)c->log_every - c->steps_done % (unsigned long long)c->log_every;
        n = std::min<long long>(n, to_step_end + (long long)(steps_to_log - 1) * ns);
      }
      CoopSchedule& sch = c->coop;
      for (int k = 0; k < ns; ++k) sch.w[k] = c->w[k];
      sch.ns = ns; sch.first = (int)(i % ns); sch.nstages = (int)n; sch.call_ends = (i + n == S) ? 1 : 0;
      sch.dt = c->dt; sch.adaptive = c->adaptive ? 1 : 0;
      st = (int)dispatch(c, OP_KICK_COOP, 0);
      if (st != PYCOOL_OK) {                                 // e.g. the GPU is shared and the grid is not co-resident:
        cudaGetLastError();                                  // nothing was launched; go on one launch per stage
        coop = false;
        c->cooperative = false;
        continue;
      }
      c->counts[0] += (unsigned long long)n;
      if (n & 1) c->cur ^= 1;
      const long long steps_ended = (i % ns + n) / ns;       // steps completed inside this launch
      i += n;
      if (c->log_every > 0 && steps_ended > 0) {
        c->steps_done += (unsigned long long)steps_ended;
        if (i % ns == 0 && c->steps_done % (unsigned long long)c->log_every == 0) {
          st = enqueue_energy(c, true, c->d_log + (c->log_n % (unsigned long long)c->log_cap));
          if (st != PYCOOL_OK) return st;
          c->log_n++;
        }
      }
      continue;
    }
    len.w = c->w[i % ns];
    len.w_next = (i + 1 < S) ? c->w[(i + 1) % ns] : 0.0;      // stage weights are never zero
    len.ends_step = (i % ns) == ns - 1;
    if (c->profiling) CUDA_TRY(c, cudaEventRecord(c->ev[c->ev_used++], c->stream));
    c->len = len;
    st = (int)dispatch(c, OP_KICK, 0);
    if (st != PYCOOL_OK) return st;
    if (c->profiling) CUDA_TRY(c, cudaEventRecord(c->ev[c->ev_used++], c->stream));
    c->counts[0]++;
    c->cur ^= 1;
    if (!c->fused_tail) {
      st = launch_scalar(c, len, 1);
      if (st != PYCOOL_OK) return st;
    }
    if (len.ends_step && c->log_every > 0 && ++c->steps_done % (unsigned long long)c->log_every == 0) {
      // energy log: a read-out of the state this step ends in (its closing half drift applied on the fly, the
      // scale factor of that instant), appended on the device; the step sequence itself is untouched
      st = enqueue_energy(c, true, c->d_log + (c->log_n % (unsigned long long)c->log_cap));
      if (st != PYCOOL_OK) return st;
      c->log_n++;
    }
    ++i;
  }
  c->pending_drift = true;
  return PYCOOL_OK;
}

int pycool_set_adaptive(pycool_ctx* c, int on) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  c->adaptive = on != 0;
  return PYCOOL_OK;
}

int pycool_flush(pycool_ctx* c) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  return ensure_flushed(c);
}

int pycool_sync(pycool_ctx* c) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (int st = ensure_flushed(c)) return st;
  Scalars s;
  return read_scalars(c, &s);
}

int pycool_read_fields(pycool_ctx* c, void* phi_host, void* pi_host) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!c->have_fields) return fail(c, PYCOOL_ESTATE, "read before set_fields");
  int st = ensure_flushed(c);
  if (st != PYCOOL_OK) return st;
  if (phi_host) st = copy_dense(c, c->phi[c->cur], phi_host, false, cudaMemcpyDeviceToHost);
  if (st == PYCOOL_OK && pi_host) st = copy_dense(c, c->pi[c->cur], pi_host, false, cudaMemcpyDeviceToHost);
  if (st != PYCOOL_OK) return st;
  Scalars s;
  return read_scalars(c, &s);
}

int pycool_read_fields_device(pycool_ctx* c, void* d_phi_dst, void* d_pi_dst) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!c->have_fields) return fail(c, PYCOOL_ESTATE, "read before set_fields");
  int st = ensure_flushed(c);
  if (st != PYCOOL_OK) return st;
  if (d_phi_dst) st = copy_dense(c, c->phi[c->cur], d_phi_dst, false, cudaMemcpyDeviceToDevice);
  if (st == PYCOOL_OK && d_pi_dst) st = copy_dense(c, c->pi[c->cur], d_pi_dst, false, cudaMemcpyDeviceToDevice);
  return st;
}

int pycool_device_fields(pycool_ctx* c, void** d_phi, void** d_pi, size_t layout[4]) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (int st = ensure_flushed(c)) return st;
  if (d_phi) *d_phi = c->phi[c->cur];
  if (d_pi) *d_pi = c->pi[c->cur];
  if (layout) {
    layout[0] = (size_t)c->lay.pitch; layout[1] = (size_t)c->lay.rows;
    layout[2] = (size_t)c->lay.gx; layout[3] = (size_t)c->lay.gy;
  }
  return PYCOOL_OK;
}

int pycool_energies(pycool_ctx* c, pycool_energy* o) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!o) return fail(c, PYCOOL_EINVAL, "out is NULL");
  if (!c->have_fields) return fail(c, PYCOOL_ESTATE, "energies before set_fields");
  return energies_now(c, o);
}

int pycool_set_energy_cadence(pycool_ctx* c, int every, int capacity) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (every < 0 || (every > 0 && capacity < 1) || capacity > (1 << 24))
    return fail(c, PYCOOL_EINVAL, "every must be >= 0 and capacity 1 .. 2^24");
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (c->d_log) cudaFree(c->d_log);
  c->d_log = nullptr;
  c->log_every = 0; c->log_cap = 0; c->log_n = 0; c->steps_done = 0;
  if (every == 0) return PYCOOL_OK;
  if (cudaMalloc(&c->d_log, (size_t)capacity * sizeof(pycool_energy)) != cudaSuccess) {
    cudaGetLastError();
    return fail(c, PYCOOL_ENOMEM, "cudaMalloc of the energy log (%d entries) failed", capacity);
  }
  c->log_every = every; c->log_cap = capacity;
  return PYCOOL_OK;
}

int pycool_read_energy_log(pycool_ctx* c, pycool_energy* out_host, int max_entries, int* n_out,
                           unsigned long long* total) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (!n_out || max_entries < 0 || (max_entries > 0 && !out_host)) return fail(c, PYCOOL_EINVAL, "bad output arguments");
  *n_out = 0;
  if (total) *total = c->log_n;
  if (!c->d_log) return PYCOOL_OK;
  const unsigned long long have = std::min<unsigned long long>(c->log_n, (unsigned long long)c->log_cap);
  const int n = (int)std::min<unsigned long long>(have, (unsigned long long)max_entries);
  // the newest n entries, oldest first; entry number j (0-based since the cadence was set) sits in slot j % capacity
  for (int i = 0; i < n; ++i) {
    const unsigned long long j = c->log_n - (unsigned long long)n + (unsigned long long)i;
    CUDA_TRY(c, cudaMemcpyAsync(out_host + i, c->d_log + (j % (unsigned long long)c->log_cap), sizeof(pycool_energy),
                                cudaMemcpyDeviceToHost, c->stream));
  }
  Scalars s;
  int st = read_scalars(c, &s);            // synchronises; reports a non-finite sum
  if (st != PYCOOL_OK) return st;
  *n_out = n;
  return PYCOOL_OK;
}

int pycool_destroy(pycool_ctx* c) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (c->stream || !c->own_stream) cudaStreamSynchronize(c->stream);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  if (c->d_log) cudaFree(c->d_log);
  if (c->own_stream) cudaStreamDestroy(c->stream);
  if (c->owned_block) cudaFree(c->owned_block);
  delete c;
  return PYCOOL_OK;
}

const char* pycool_last_error(const pycool_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

int pycool_stage_weights(int order, double* w, int cap) {
  long double t[16];
  const int s = stage_weights_ld(order, t);
  if (s == 0 || !w || cap < s) return 0;
  for (int i = 0; i < s; ++i) w[i] = (double)t[i];
  return s;
}

int pycool_launch_counts(const pycool_ctx* c, unsigned long long counts[4]) {
  if (!c || !counts) return PYCOOL_EINVAL;
  for (int i = 0; i < 4; ++i) counts[i] = c->counts[i];
  return PYCOOL_OK;
}

int pycool_set_profiling(pycool_ctx* c, int on) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  c->profiling = on != 0;
  c->ev_used = 0; c->prof_ms = 0; c->prof_n = 0;
  return PYCOOL_OK;
}

int pycool_kick_time_ms(pycool_ctx* c, double* total_ms, unsigned long long* launches) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
    float ms = 0;
    CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
    c->prof_ms += ms;
    c->prof_n++;
  }
  c->ev_used = 0;
  if (total_ms) *total_ms = c->prof_ms;
  if (launches) *launches = c->prof_n;
  return PYCOOL_OK;
}

int pycool_kick_geometry(const pycool_ctx* c, int tile[10]) {
  if (!c || !tile) return PYCOOL_EINVAL;
  const TileInfo& t = kTiles[c->tile];
  tile[0] = t.tx; tile[1] = t.ty; tile[2] = c->zc; tile[3] = t.nt;
  tile[4] = (int)(c->grid.x * c->grid.y * c->grid.z);
  tile[5] = (int)dispatch(const_cast<pycool_ctx*>(c), OP_SMEM, c->tile);
  tile[6] = c->tile;
  tile[7] = t.stages;
  tile[8] = c->region[0]; tile[9] = c->region[1];
  return PYCOOL_OK;
}

int pycool_set_zchunk(pycool_ctx* c, int planes) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (planes < 0) return fail(c, PYCOOL_EINVAL, "planes < 0");
  c->zc_user = planes;
  return set_geometry(c);
}

int pycool_set_item_order(pycool_ctx* c, int tiles_per_region) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (tiles_per_region < -1) return fail(c, PYCOOL_EINVAL, "tiles_per_region must be -1 (automatic), 0 (plain order) or > 0");
  c->region_user = tiles_per_region;
  return set_geometry(c);
}

int pycool_set_overlap(pycool_ctx* c, int on) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  c->overlap_launch = on != 0;
  return PYCOOL_OK;
}

int pycool_set_energy_kernel(pycool_ctx* c, int tma) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (tma < 0 || tma > 4) return fail(c, PYCOOL_EINVAL, "energy kernel must be 0 (plain), 1 (automatic) or 2..4 (a TMA variant)");
  c->energy_tma = tma;
  return PYCOOL_OK;
}

int pycool_set_persistent(pycool_ctx* c, int on) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  c->persistent = on != 0;
  return PYCOOL_OK;
}

int pycool_set_cooperative(pycool_ctx* c, int on) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  c->cooperative = on != 0;
  return PYCOOL_OK;
}

int pycool_set_fused_tail(pycool_ctx* c, int on) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  c->fused_tail = on != 0;
  return PYCOOL_OK;
}

int pycool_set_tile(pycool_ctx* c, int tile) {
  if (!c) return PYCOOL_EINVAL;
  OnDevice on_device(c);
  if (tile < -1 || tile >= kNumTiles) return fail(c, PYCOOL_EINVAL, "tile must be -1 (auto) .. %d", kNumTiles - 1);
  if (tile >= 0 && !tile_allowed(c->lay, tile))
    return fail(c, PYCOOL_EINVAL, "tile %d is a TMA variant: it needs the ghost layout (even N >= 4; N %% 4 == 0 for x quads)", tile);
  if (tile >= 0 && (size_t)dispatch(c, OP_SMEM, tile) > kMaxSmem)
    return fail(c, PYCOOL_EINVAL, "tile %d needs %zu bytes of shared memory for this model and precision (limit %zu)",
                tile, (size_t)dispatch(c, OP_SMEM, tile), kMaxSmem);
  if (tile >= 0 && !dispatch(c, OP_BUILT, tile))
    return fail(c, PYCOOL_EINVAL, "tile %d is not built for %d fields at this precision (register budget)", tile, c->nf);
  c->tile = tile < 0 ? auto_tile(c) : tile;
  return set_geometry(c);
}

}  // extern "C"
