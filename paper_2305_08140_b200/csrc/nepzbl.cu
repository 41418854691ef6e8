// nepzbl.cu -- host side of the C ABI declared in include/nepzbl.h: parameter upload, workspace
// carving, kernel sequencing on one CUDA stream.  All arithmetic of the path runs in the kernels
// of neighbor.cuh / descriptor.cuh / force.cuh / integrate.cuh.  No CPU fallback exists.
#include "nepzbl.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <type_traits>
#include <vector>

#include "common.cuh"
#include "neighbor.cuh"
#include "descriptor.cuh"
#include "descriptor_split.cuh"
#include "descriptor_tc.cuh"
#include "descriptor_split_tc.cuh"
#include "force.cuh"
#include "site_fp64.cuh"
#include "integrate.cuh"
#include "wigner_seitz.cuh"

namespace {

thread_local std::string g_create_error;

constexpr int kTraceRing = 1024;

struct Carve {  // byte offsets into the workspace
  size_t xyzt, xyzt_build, xyzt_tmp, perm, inv_perm, order, cell_of, cell_count, cell_fill, cell_start, scan_sum, scan_off,
      nn_r, nn_a, shellq, nl_r, rev, rmask, tmask, amask, adisp, q_radial, dk, pforce, u_site, q_desc, zbl_list, dense_list, tiles, nl_loc, md_force, md_energy,
      partial, nhc_partial, st_pos, st_types, st_e, st_f, st_w, total;
  int npad, ncell_cap;
};

struct ShapeId {
  int nr, kr, na, ka, b4, nt, b5;
};

}  // namespace

struct nepzbl_handle {
  nepzbl_params p{};  // scalar fields only (pointers nulled)
  int D = 0, shape = -1;      // D: descriptor components of the kernel shape
  int D_model = 0;            // ... of the caller's model (smaller when the model runs zero-padded on a larger shape)
  bool padded = false;
  std::vector<int> qmap;      // model component -> shape component
  int* d_qmap = nullptr;
  int device = 0;
  cudaStream_t stream = nullptr;
  cudaStream_t own_stream = nullptr;  // created when the caller passes no stream (see nep_zbl_create)
  std::string err;
  std::string graph_note;             // why MD steps are not replayed as a graph (empty: they are)
  long long launches = 0;

  // library-owned small device block
  Scalars* d_sc = nullptr;
  BoxMap* d_bm = nullptr;
  float* d_nnw = nullptr;
  double* d_mass = nullptr;
  double* d_inv_mass = nullptr;
  double* d_trace = nullptr;  // [kTraceRing]
  double* d_esum = nullptr;   // [2]
  Scalars* h_sc = nullptr;    // pinned
  double* h_trace = nullptr;  // pinned [kTraceRing]
  double* h_esum = nullptr;   // pinned [2]
  std::vector<char> tables;   // ModelTables<MS> for the dispatched shape
  ZblParams zp{};
  SiteModel site{};           // fp64 tables of k_site_fp64 (d_site holds them)
  double* d_site = nullptr;
  // network layer: 0 = CUDA cores (FFMA, k_angular_nn), 1 = mma.sync 3xTF32, 2 = tcgen05 3xTF32 inside k_angular_nn
  // (block-synchronous), 3 = k_angular_tc (descriptor_tc.cuh: tcgen05, software-pipelined over two tiles).
  // NEPZBL_NN=ffma|mma|tcsync|tc overrides the default; measured verdict in DESIGN.md / profiles/r2_nn_tensor.md
  int nn_mode = 3;
  bool split_tc = false;      // four-lane models: k_angular_split_tc instead of k_angular_nn_split (nn_mode 3, <= 104 neurons)
  bool dense_on = true;       // NEPZBL_DENSE_THRESHOLD=off disables the fp64 re-evaluation (measurement aid)
  size_t smem_nn = 0;
  // threads per block of k_radial / k_force: one warp while the grid is only a few waves of resident threads (the
  // partly filled last wave costs one block's duration: 128 000 atoms 32: 78.3 us, 64: 80.5, 128: 83.1 for
  // k_force), two warps beyond (8.192 M atoms 32: 4.17 ms, 64: 4.02, 128: 4.11).  NEPZBL_GATHER_BLOCK overrides.
  int gather_block = 0;
  int n_sm = 0, ang_grid = 0;  // k_angular_nn is persistent: grid = resident blocks

  // workspace
  char* ws = nullptr;
  size_t ws_bytes = 0;
  long long n_cap = 0;
  Carve cv{};

  // list state
  bool have_list = false;
  long long n = 0;
  double box[9] = {0};
  int pbc[3] = {0, 0, 0};
  bool tri = false;            // triclinic box (all axes periodic): box_inv / box_hgt are set
  double box_inv[9] = {0}, box_hgt[3] = {0};

  // md state
  bool md_ready = false;
  double* md_pos = nullptr;
  double* md_vel = nullptr;
  const int32_t* md_types = nullptr;
  long long md_steps = 0;

  // Nose-Hoover chain on a group of atoms (md_set_thermostat)
  NhcState* d_nhc = nullptr;
  NhcState* h_nhc = nullptr;              // pinned
  const unsigned char* md_group = nullptr;  // dev, caller-owned
  bool nhc_on = false;

  // Wigner-Seitz reference (library-owned device arrays, freed at destroy)
  struct {
    long long ns = 0;
    WsGrid g{};
    int *cell_of = nullptr, *cell_count = nullptr, *cell_fill = nullptr, *cell_start = nullptr, *occ = nullptr;
    WsSite* rec = nullptr;                // cell-sorted {x, y, z, index}
    unsigned long long* out = nullptr;    // dev [8]: bounds / counts
    unsigned long long* h_out = nullptr;  // pinned [8]
  } ws_ref;

  // one MD step captured as a CUDA graph: the list-rebuild chain and the ZBL kernel sit in IF nodes
  // whose conditions are set on the device (last block of k_kick_drift / k_force), so a step is ONE launch
  cudaGraph_t step_graph = nullptr;
  cudaGraphExec_t step_exec = nullptr;
  cudaStream_t cap_stream = nullptr;
  // md_step_host: the positions are final once k_kick_drift has run, so their device-to-host copy goes to a
  // second stream behind this event and overlaps the force kernels
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_drift = nullptr;
  int graph_kernels = 0, graph_rebuild_kernels = 0;  // launch accounting per graph replay
  bool use_graph = true;

  // per-kernel CUDA-event timing (nep_zbl_profile)
  bool prof = false;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0;
  struct Span { int id; cudaEvent_t a, b; };
  std::vector<Span> spans;
  cudaEvent_t ev_open = nullptr;
  int ev_open_id = -1;

  template <class T>
  T* at(size_t off) const { return reinterpret_cast<T*>(ws + off); }
};

namespace {

int fail(nepzbl_handle* h, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (h) h->err = buf; else g_create_error = buf;
  return code;
}

#define CU(call)                                                                             \
  do {                                                                                       \
    cudaError_t e_ = (call);                                                                 \
    if (e_ != cudaSuccess)                                                                   \
      return fail(h, NEPZBL_E_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                  __FILE__, __LINE__);                                                       \
  } while (0)

inline size_t al(size_t x) { return (x + 255) & ~size_t(255); }

// 32-bit words of the per-lane in-cutoff mask: lane p of RADIAL_LANES owns entries p, p+4, ...
inline int mask_words(const nepzbl_params& p) { return (p.cap_radial + 32 * RADIAL_LANES - 1) / (32 * RADIAL_LANES); }

// 64-bit words of the angular in-cutoff mask per atom (cap_angular <= 128)
inline int amask_words(const nepzbl_params& p) { return (p.cap_angular + 63) / 64; }

// NEPZBL_STAGE=1|2: neighbour tiles staged in shared memory by k_radial (stage.cuh; measurement aid, default off)
inline int stage_mode() {
  static const int m = [] { const char* e = getenv("NEPZBL_STAGE"); const int v = e ? atoi(e) : 0; return v == 1 || v == 2 ? v : 0; }();
  return m;
}

Carve carve(const nepzbl_params& p, int D, long long n_cap) {
  Carve c{};
  long long npad = (n_cap + 127) / 128 * 128;
  if (npad < 128) npad = 128;
  c.npad = (int)npad;
  c.ncell_cap = (int)(n_cap + 8192);  // half-size cells hold ~2.7 atoms in bcc W
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o = al(o + bytes); return r; };
  c.xyzt = take(16 * npad);
  c.xyzt_build = take(16 * npad);
  c.xyzt_tmp = take(16 * npad);
  c.perm = take(4 * npad);
  c.inv_perm = take(4 * npad);
  c.order = take(4 * npad);
  c.cell_of = take(4 * npad);
  c.cell_count = take(4 * ((size_t)c.ncell_cap + 1));
  c.cell_fill = take(4 * ((size_t)c.ncell_cap + 1));
  c.cell_start = take(4 * ((size_t)c.ncell_cap + 1));
  c.scan_sum = take(4 * ((size_t)c.ncell_cap / SCAN_TILE + 2));  // tile totals / offsets of the cell scan
  c.scan_off = take(4 * ((size_t)c.ncell_cap / SCAN_TILE + 2));
  c.nn_r = take(4 * npad);
  c.nn_a = take(4 * npad);
  c.shellq = take(8 * npad);
  c.nl_r = take(4 * (size_t)((p.cap_radial + 3) / 4 * 4) * npad);  // whole groups of four rows (nl_at)
  c.rev = take((size_t)p.cap_angular * npad);
  c.rmask = take(4 * (size_t)mask_words(p) * RADIAL_LANES * npad);
  c.tmask = p.n_types > 1 ? take(4 * (size_t)mask_words(p) * RADIAL_LANES * npad) : c.rmask;  // types of the in-cutoff entries
  c.amask = take(8 * (size_t)amask_words(p) * npad);
  c.adisp = take(16 * (size_t)p.cap_angular * npad);
  c.q_radial = take(4 * (size_t)(p.n_max_radial + 1) * npad);
  c.dk = take(64 * (size_t)std::max(1, p.n_types) * npad);  // AtomRec, one per partner type
  c.pforce = take(16 * (size_t)p.cap_angular * npad);
  c.u_site = take(4 * npad);
  c.q_desc = take(4 * (size_t)D * npad);
  c.zbl_list = take(4 * npad);
  c.dense_list = take(4 * npad);
  if (stage_mode() > 0) {  // neighbour-tile staging experiment (stage.cuh)
    c.tiles = take(sizeof(TileDesc) * (size_t)(npad / STAGE_TILE + 1));
    c.nl_loc = take(2 * (size_t)p.cap_radial * npad);
  }
  c.md_force = take(12 * npad);
  c.md_energy = take(8 * npad);
  c.partial = take(16 * 1024);
  c.nhc_partial = take(16 * 1024);  // [1024] sums + [1024] counts
  c.st_pos = take(24 * npad);
  c.st_types = take(4 * npad);
  c.st_e = take(8 * npad);
  c.st_f = take(12 * npad);
  c.st_w = take(36 * npad);
  c.total = o;
  return c;
}

// instantiated model shapes: BASELINE.json configs (with / without the 4-body term) and the paper's own
// sizes (n_max 15 / 10, l_max 4; basis 8 / 8 is DESIGN.md C-26) -- SURVEY 8(f) NEXT-2
// Any model that FITS one of them runs on it (nep_zbl_create pads its tables with zeros: a channel whose coefficients are
// zero has zero descriptor components, and their columns of w0 are zero too), so the sizes really are run-time
// parameters within n_max <= 15 / 10 and basis <= 8; the table lists exact matches first, then by cost.
const ShapeId kShapes[] = {{5, 9, 5, 9, 1, 1, 0}, {5, 9, 5, 9, 0, 1, 0}, {16, 9, 11, 9, 0, 1, 0}, {5, 9, 5, 9, 1, 2, 0},
                           {5, 9, 5, 9, 1, 1, 1}, {16, 9, 11, 9, 0, 2, 0}, {16, 9, 11, 9, 1, 1, 0}};
// order in which a model that matches none exactly looks for a shape that contains it (cheapest first)
const int kShapeByCost[] = {1, 0, 4, 3, 2, 6, 5};
using MS0 = ModelShape<5, 9, 5, 9, true>;
using MS1 = ModelShape<5, 9, 5, 9, false>;
using MS2 = ModelShape<16, 9, 11, 9, false>;
using MS3 = ModelShape<5, 9, 5, 9, true, 2>;         // two atom types
using MS4 = ModelShape<5, 9, 5, 9, true, 1, true>;   // 4-body + 5-body terms (NEXT-4, C-27)
using MS5 = ModelShape<16, 9, 11, 9, false, 2>;      // paper-sized model with two atom types (NEXT-4)
using MS6 = ModelShape<16, 9, 11, 9, true>;          // paper-sized channels with the 4-body term (hosts padded models)
template <class F>
void with_shape(int shape, F&& f) {
  switch (shape) {
    case 0: f(MS0{}); break;
    case 1: f(MS1{}); break;
    case 2: f(MS2{}); break;
    case 3: f(MS3{}); break;
    case 4: f(MS4{}); break;
    case 5: f(MS5{}); break;
    default: f(MS6{}); break;
  }
}
// models with more than 5 angular channels use the four-lanes-per-atom kernel (descriptor_split.cuh)
template <class MS>
constexpr bool kSplit = MS::NA > 5;
// ... and its tensor-core form (descriptor_split_tc.cuh) when the slices are 16 entries (no 4-/5-body term)
template <class MS>
constexpr bool kSplitTc = kSplit<MS> && !MS::B4 && !MS::B5 && SplitLayout<MS>::SLP == 16;

// canonical descriptor index (SURVEY 8(c) C order) of a component in a model with nr radial / na angular channels:
// block 0 radial n; blocks 1..4 the 3-body l; block 5 the 4-body term; block 6 the 5-body term (behind the 4-body one)
inline int desc_index(int nr, int na, bool b4, int block, int n) {
  if (block == 0) return n;
  if (block <= 4) return nr + (block - 1) * na + n;
  if (block == 5) return nr + 4 * na + n;
  return nr + 4 * na + (b4 ? na : 0) + n;
}

template <class MS>
void build_tables(nepzbl_handle* h, const nepzbl_params* p) {
  ModelTables<MS> t;
  memset(&t, 0, sizeof t);
  auto fold = [](const double* c, int N, int K, float* ct, float* kct) {
    for (int n = 0; n < N; ++n) {
      double s = 0.0;
      for (int k = 1; k < K; ++k) s += c[n * K + k];
      for (int k = 0; k < K; ++k) {
        double v = k == 0 ? c[n * K] + 0.5 * s : 0.5 * c[n * K + k];
        ct[n * K + k] = (float)v;
        if (kct) kct[n * K + k] = (float)(k * v);
      }
    }
  };
  for (int pr = 0; pr < MS::NT * MS::NT; ++pr) {  // params: [ti][tj][n][k]
    fold(p->c_radial + (size_t)pr * MS::NR * MS::KR, MS::NR, MS::KR, &t.ctR[pr][0][0], nullptr);
    fold(p->c_angular + (size_t)pr * MS::NA * MS::KA, MS::NA, MS::KA, &t.ctA[pr][0][0], &t.kctA[pr][0][0]);
  }
  t.inv_rcR = (float)(1.0 / p->rc_radial);
  t.inv_rcA = (float)(1.0 / p->rc_angular);
  t.rcR2 = (float)(p->rc_radial * p->rc_radial);
  t.rcA2 = (float)(p->rc_angular * p->rc_angular);
  double zf = p->zbl_r_outer + 0.01;
  t.zbl_flag_r2 = p->zbl_enabled ? (float)(zf * zf) : 0.0f;
  t.inv_shell_w = p->skin > 0 ? (float)(8.0 / p->skin) : 0.0f;
  t.b1 = (float)p->b1;
  t.n_neurons = p->n_neurons;
  // fp64 re-evaluation thresholds on the angular network inputs |s q| (site_fp64.cuh):
  // 8 for the 3-body inputs, 3 for the 4-/5-body inputs.  A 300 K crystal stays below 0.8 / 0.4 and the atoms of a free
  // (001) surface below 6.2 / 1.3 (coherent l = 1 sums, accurate in fp32), so neither is listed; the disordered
  // sites that miss the tolerance in fp32 have 4-body inputs of 50-2500.  NEPZBL_DENSE_THRESHOLD overrides: "off",
  // one number (both thresholds) or "t3,t4".
  t.dense_thr = 8.0f;
  t.dense_thr4 = 3.0f;
  if (const char* dt = getenv("NEPZBL_DENSE_THRESHOLD")) {
    if (!strcmp(dt, "off")) h->dense_on = false;
    else if (atof(dt) > 0.0) {
      t.dense_thr = t.dense_thr4 = (float)atof(dt);
      if (const char* comma = strchr(dt, ','))
        if (atof(comma + 1) > 0.0) t.dense_thr4 = (float)atof(comma + 1);
    }
  }
  h->tables.resize(sizeof t);
  memcpy(h->tables.data(), &t, sizeof t);
  if (kSplit<MS>) {
    using LY = SplitLayout<MS>;
    h->smem_nn = sizeof(float) * ((size_t)LY::table_floats(LY::rows(p->n_neurons)) + LY::stash_floats());
    h->split_tc = false;
    if constexpr (kSplitTc<MS>) {
      h->split_tc = h->nn_mode == 3 && p->n_neurons <= STC_KT;
      if (h->split_tc) h->smem_nn = StcLayout<MS>::smem_bytes(LY::rows(p->n_neurons));
    }
  } else {
    const size_t nrow = (size_t)nn_rows(p->n_neurons);
    h->smem_nn = sizeof(float) * (nrow * MS::DPAD + 2 * nrow + MS::DPAD);
    if (MS::NT > 1) h->smem_nn += sizeof(float) * (2 * MS::NT * MS::NT * MS::NA * CT_ROW);
    if (h->nn_mode >= 2 && p->n_neurons > TC_NP - 8) h->nn_mode = 0;  // the tcgen05 variants hold at most 56 neurons
    if (h->nn_mode == 1) h->smem_nn += sizeof(float) * (32 * ((MS::D + 7) / 8 * 8 + 4) + 32);  // X / Fp tile and site energies
    if (h->nn_mode >= 2) h->smem_nn += tc_smem_bytes<MS>();
  }
}

// folded Chebyshev coefficients (descriptor.cuh): ct_n0 = c_n0 + 1/2 sum_{k>=1} c_nk, ct_nk = c_nk / 2
inline double folded(const double* c, int K, int n, int k) {
  if (k > 0) return 0.5 * c[n * K + k];
  double s = 0.0;
  for (int j = 1; j < K; ++j) s += c[n * K + j];
  return c[n * K] + 0.5 * s;
}

template <class MS>
std::vector<float> build_nnw(const nepzbl_params* p) {
  if constexpr (kSplit<MS>) {
    // table of k_angular_nn_split, in the order SplitLayout::table_floats lists (weights and q_scaler permuted
    // into the four lane slices; everything not written stays zero)
    using LY = SplitLayout<MS>;
    const int nrow = LY::rows(p->n_neurons);
    std::vector<float> w((size_t)LY::table_floats(nrow), 0.0f);
    float* w0 = w.data();
    float* b0 = w0 + (size_t)nrow * 4 * LY::SLS;
    float* w1 = b0 + nrow;
    float* qs = w1 + nrow;
    float* cta = qs + 4 * LY::SLS;
    float* ctr = cta + LY::NPR * LY::NAP * MS::KA;
    for (int lane = 0; lane < 4; ++lane)
      for (int idx = 0; idx < LY::SLP; ++idx) {
        const int nu = LY::nu(lane, idx);
        if (nu < 0) continue;
        qs[lane * LY::SLS + idx] = (float)p->q_scaler[nu];
        for (int m = 0; m < p->n_neurons; ++m)
          w0[((size_t)m * 4 + lane) * LY::SLS + idx] = (float)p->w0[(size_t)m * MS::D + nu];
      }
    for (int m = 0; m < p->n_neurons; ++m) {
      b0[m] = (float)p->b0[m];
      w1[m] = (float)p->w1[m];
    }
    for (int pr = 0; pr < LY::NPR; ++pr) {  // params: [ti][tj][n][k]
      for (int nq = 0; nq < MS::NA; ++nq)
        for (int k = 0; k < MS::KA; ++k)
          cta[((size_t)pr * LY::NAP + nq) * MS::KA + k] = (float)folded(p->c_angular + (size_t)pr * MS::NA * MS::KA, MS::KA, nq, k);
      for (int nq = 0; nq < MS::NR; ++nq)
        for (int k = 0; k < MS::KR; ++k)
          ctr[((size_t)pr * 4 * LY::RSUB + nq) * MS::KR + k] = (float)folded(p->c_radial + (size_t)pr * MS::NR * MS::KR, MS::KR, nq, k);
    }
    // k_angular_split_tc: behind the table (next multiple of 32 floats) the B operands of its two products, tf32 hi + lo,
    // tiled as tc05.cuh describes: B1 hi/lo [112 neurons][64 = 4 slices x 16], B2 hi/lo [64][104 neurons] (B1 transposed)
    if constexpr (kSplitTc<MS>) {
      if (p->n_neurons <= STC_KT) {
        const size_t off = (w.size() + 31) / 32 * 32;
        w.resize(off + 2 * (size_t)STC_NP * STC_KX + 2 * (size_t)STC_KX * STC_KT, 0.0f);
        float* b1h = w.data() + off;
        float* b1l = b1h + STC_NP * STC_KX;
        float* b2h = b1l + STC_NP * STC_KX;
        float* b2l = b2h + STC_KX * STC_KT;
        auto split = [](float x, float& hi, float& lo) {  // round to nearest tf32 (13 low bits cleared), remainder
          uint32_t u;
          memcpy(&u, &x, 4);
          u = (u + 0x1000u) & 0xFFFFE000u;
          memcpy(&hi, &u, 4);
          lo = x - hi;
        };
        for (int lane = 0; lane < 4; ++lane)
          for (int idx = 0; idx < LY::SLP; ++idx) {
            const int nu = LY::nu(lane, idx);
            if (nu < 0) continue;
            const int v = LY::SLP * lane + idx;
            for (int m = 0; m < p->n_neurons; ++m) {
              const float x = (float)p->w0[(size_t)m * MS::D + nu];
              const size_t o1 = tc05::tile_off(STC_NP, m, v) / 4, o2 = tc05::tile_off(STC_KX, v, m) / 4;
              split(x, b1h[o1], b1l[o1]);
              split(x, b2h[o2], b2l[o2]);
            }
          }
      }
    }
    return w;
  } else {
    const int neu2 = nn_rows(p->n_neurons);  // zero padding rows, see nn_rows
    const size_t ct_floats = MS::NT > 1 ? 2 * MS::NT * MS::NT * MS::NA * CT_ROW : 0;  // rows padded to CT_ROW floats
    std::vector<float> w((size_t)neu2 * MS::DPAD + 2 * neu2 + MS::DPAD + ct_floats, 0.0f);
    for (int m = 0; m < p->n_neurons; ++m)
      for (int v = 0; v < MS::D; ++v) w[(size_t)m * MS::DPAD + v] = (float)p->w0[(size_t)m * MS::D + v];
    float* b0 = w.data() + (size_t)neu2 * MS::DPAD;
    float* w1 = b0 + neu2;
    float* qs = w1 + neu2;
    for (int m = 0; m < p->n_neurons; ++m) {
      b0[m] = (float)p->b0[m];
      w1[m] = (float)p->w1[m];
    }
    for (int v = 0; v < MS::D; ++v) qs[v] = (float)p->q_scaler[v];
    if (MS::NT > 1) {  // ct [NT*NT][NA][KA], then k * ct (k_angular_nn reads them from shared memory)
      float* ct = qs + MS::DPAD;
      for (int pr = 0; pr < MS::NT * MS::NT; ++pr)
        for (int nq = 0; nq < MS::NA; ++nq)
          for (int k = 0; k < MS::KA; ++k) {
            const double v = folded(p->c_angular + (size_t)pr * MS::NA * MS::KA, MS::KA, nq, k);
            ct[(pr * MS::NA + nq) * CT_ROW + k] = (float)v;
            ct[((MS::NT * MS::NT + pr) * MS::NA + nq) * CT_ROW + k] = (float)(k * v);
          }
    }
    // k_angular_tc: behind the table (at the next multiple of 32 floats) the B operands of its two tensor-core products,
    // split into tf32 hi + lo parts and laid out as the tiles tc05.cuh describes:
    //   B1 hi/lo [64 neurons][kp]: w0 with -b0 in column D;  B2 hi/lo [kn components][64 neurons]: w0 transposed
    if (p->n_neurons <= TC_NP - 8) {
      constexpr TcShape ts = tc_shape<MS>();
      const size_t off = (w.size() + 31) / 32 * 32;
      w.resize(off + 2 * (size_t)TC_NP * ts.kp + 2 * (size_t)ts.kn * TC_NP, 0.0f);
      float* b1h = w.data() + off;
      float* b1l = b1h + TC_NP * ts.kp;
      float* b2h = b1l + TC_NP * ts.kp;
      float* b2l = b2h + ts.kn * TC_NP;
      auto split = [](float x, float& hi, float& lo) {  // cvt.rna.tf32: nearest, ties away from zero, 13 low bits cleared
        uint32_t u;
        memcpy(&u, &x, 4);
        u = (u + 0x1000u) & 0xFFFFE000u;
        memcpy(&hi, &u, 4);
        lo = x - hi;
      };
      for (int m = 0; m < p->n_neurons; ++m) {
        for (int k = 0; k <= MS::D; ++k) {
          const float x = k < MS::D ? (float)p->w0[(size_t)m * MS::D + k] : -(float)p->b0[m];
          const size_t o = tc05::tile_off(TC_NP, m, k) / 4;
          split(x, b1h[o], b1l[o]);
        }
        for (int v = 0; v < MS::D; ++v) {
          const size_t o = tc05::tile_off(ts.kn, v, m) / 4;
          split((float)p->w0[(size_t)m * MS::D + v], b2h[o], b2l[o]);
        }
      }
    }
    return w;
  }
}

// fp64 tables of k_site_fp64: folded Chebyshev coefficients, q_scaler, network weights (one device buffer)
template <class MS>
std::vector<double> build_site_tables(const nepzbl_params* p, SiteModel* sm, size_t off[6]) {
  sm->NT = MS::NT; sm->NR = MS::NR; sm->KR = MS::KR; sm->NA = MS::NA; sm->KA = MS::KA; sm->B4 = MS::B4 ? 1 : 0;
  sm->B5 = MS::B5 ? 1 : 0;
  sm->D = MS::D; sm->n_neurons = p->n_neurons; sm->fprec = MS::FPREC ? 1 : 0;
  sm->b1 = p->b1; sm->rcA = p->rc_angular;
  const int npr = MS::NT * MS::NT;
  std::vector<double> v;
  off[0] = v.size();
  for (int pr = 0; pr < npr; ++pr)
    for (int nq = 0; nq < MS::NA; ++nq)
      for (int k = 0; k < MS::KA; ++k) v.push_back(folded(p->c_angular + (size_t)pr * MS::NA * MS::KA, MS::KA, nq, k));
  off[1] = v.size();
  for (int pr = 0; pr < npr; ++pr)
    for (int nq = 0; nq < MS::NR; ++nq)
      for (int k = 0; k < MS::KR; ++k) v.push_back(folded(p->c_radial + (size_t)pr * MS::NR * MS::KR, MS::KR, nq, k));
  off[2] = v.size();
  for (int d = 0; d < MS::D; ++d) v.push_back(p->q_scaler[d]);
  off[3] = v.size();
  for (size_t k = 0; k < (size_t)p->n_neurons * MS::D; ++k) v.push_back(p->w0[k]);
  off[4] = v.size();
  for (int m = 0; m < p->n_neurons; ++m) v.push_back(p->b0[m]);
  off[5] = v.size();
  for (int m = 0; m < p->n_neurons; ++m) v.push_back(p->w1[m]);
  return v;
}

inline int blocks(long long n, int b) { return (int)((n + b - 1) / b); }
// k_zbl walks the flagged atoms grid-stride: a handful in a thermal crystal (the graph skips the node when
// there is none), thousands in a cascade core, so the grid covers the device
inline int zbl_grid(const nepzbl_handle* h) { return std::max(1, std::min(blocks(h->n, 64), 8 * h->n_sm)); }

enum { PK_INTEGRATE_A = 0, PK_REBUILD, PK_RADIAL, PK_ANGULAR_NN, PK_FORCE, PK_ZBL, PK_KICK, PK_SITE64, PK_COUNT };

cudaEvent_t prof_event(nepzbl_handle* h) {
  if (h->ev_used == h->ev_pool.size()) {
    cudaEvent_t e;
    cudaEventCreate(&e);
    h->ev_pool.push_back(e);
  }
  return h->ev_pool[h->ev_used++];
}
// open a timed span for kernel group `id` (closes the previous one): events on the launch stream
void prof_mark(nepzbl_handle* h, int id) {
  if (!h->prof) return;
  cudaEvent_t e = prof_event(h);
  cudaEventRecord(e, h->stream);
  if (h->ev_open_id >= 0) h->spans.push_back({h->ev_open_id, h->ev_open, e});
  h->ev_open = e;
  h->ev_open_id = id;
}

// ------------------------------------------------------------------ kernel sequences

// S2 chain; every kernel exits immediately unless Scalars::do_rebuild is set.
int enqueue_rebuild(nepzbl_handle* h, const double* pos, const int32_t* types, cudaStream_t st) {
  const Carve& c = h->cv;
  const int n = (int)h->n, npad = c.npad;
  int nk = 0;
  BoxHost bh;
  for (int a = 0; a < 3; ++a) {
    bh.L[a] = h->box[4 * a];
    bh.pbc[a] = h->pbc[a];
  }
  bh.rcs = h->p.rc_radial + h->p.skin;
  bh.ncell_cap = c.ncell_cap;
  bh.tri = h->tri ? 1 : 0;
  for (int k = 0; k < 9; ++k) {
    bh.H[k] = h->box[k];
    bh.Hi[k] = h->box_inv[k];
  }
  for (int a = 0; a < 3; ++a) bh.hgt[a] = h->box_hgt[a];
  float rr = (float)(bh.rcs * bh.rcs);
  float rc2 = (float)(h->p.rc_radial * h->p.rc_radial);
  double ra = h->p.rc_angular + h->p.skin;
  float ra2 = (float)(ra * ra);
  k_rebuild_begin<<<1, 1, 0, st>>>(h->d_sc);
  nk++;
  if (!(h->pbc[0] && h->pbc[1] && h->pbc[2])) {
    k_bounds<<<blocks(n, 256), 256, 0, st>>>(h->d_sc, n, pos, !h->pbc[0], !h->pbc[1], !h->pbc[2]);
    nk++;
  }
  k_boxmap<<<1, 1, 0, st>>>(h->d_sc, h->d_bm, bh);
  k_zero_cells<<<blocks(c.ncell_cap + 1, 256), 256, 0, st>>>(h->d_sc, h->d_bm, h->at<int>(c.cell_count),
                                                           h->at<int>(c.cell_fill), c.ncell_cap);
  k_bin<<<blocks(n, 256), 256, 0, st>>>(h->d_sc, h->d_bm, n, pos, types, h->p.n_types, h->at<int4>(c.xyzt_tmp),
                                       h->at<int>(c.cell_of), h->at<int>(c.cell_count));
  const int scan_tiles = c.ncell_cap / SCAN_TILE + 1;
  k_scan_sums<<<scan_tiles, 1024, 0, st>>>(h->d_sc, h->d_bm, h->at<int>(c.cell_count), h->at<int>(c.scan_sum));
  k_scan_tiles<<<1, 1024, 0, st>>>(h->d_sc, h->d_bm, h->at<int>(c.scan_sum), h->at<int>(c.scan_off));
  k_scan_apply<<<scan_tiles, 1024, 0, st>>>(h->d_sc, h->d_bm, h->at<int>(c.cell_count), h->at<int>(c.scan_off),
                                            h->at<int>(c.cell_start));
  k_place<<<blocks(n, 256), 256, 0, st>>>(h->d_sc, n, h->at<int>(c.cell_of), h->at<int>(c.cell_start),
                                         h->at<int>(c.cell_fill), h->at<int>(c.order));
  k_sortcell<<<blocks(c.ncell_cap, 128), 128, 0, st>>>(h->d_sc, h->d_bm, h->at<int>(c.cell_start),
                                                      h->at<int>(c.order));
  k_permute<<<blocks(n, 256), 256, 0, st>>>(h->d_sc, n, h->at<int>(c.order), h->at<int4>(c.xyzt_tmp),
                                           h->at<int>(c.perm), h->at<int>(c.inv_perm),
                                           h->at<int4>(c.xyzt), h->at<int4>(c.xyzt_build));
  k_nbr<<<blocks(n, 128), 128, 0, st>>>(h->d_sc, h->d_bm, n, npad, h->at<int4>(c.xyzt),
                                       h->at<int>(c.cell_start), rc2, rr, ra2, h->p.cap_radial,
                                       h->p.cap_angular, h->at<int>(c.nn_r), h->at<int>(c.nl_r),
                                       h->at<int>(c.nn_a), h->at<unsigned long long>(c.shellq),
                                       (float)h->p.rc_radial, (float)(h->p.skin / 8.0));
  k_rev<<<blocks(n, 128), 128, 0, st>>>(h->d_sc, n, npad, h->at<int>(c.nn_a), h->at<int>(c.nl_r),
                                       h->at<unsigned char>(c.rev));
  if (stage_mode() > 0) {
    k_tiles<<<blocks(n, STAGE_TILE), STAGE_TILE, 0, st>>>(h->d_sc, h->d_bm, n, npad, h->at<int>(c.perm), h->at<int>(c.cell_of),
                                                         h->at<int>(c.cell_start), h->at<int>(c.nn_r), h->at<int>(c.nl_r),
                                                         h->at<TileDesc>(c.tiles), h->at<unsigned short>(c.nl_loc));
    nk++;
  }
  return nk + 11;
}

// fp64 re-evaluation of the atoms k_angular_nn listed (site_fp64.cuh); grid-stride over the list
void launch_site_fp64(nepzbl_handle* h, const double* pos, bool want_q, cudaStream_t st) {
  const Carve& c = h->cv;
  const int n = (int)h->n;
  const int grid = std::max(1, std::min(blocks(n, SITE64_WARPS), 8 * h->n_sm));
  const size_t smem = sizeof(double) * SITE64_WARPS * (2 * (size_t)h->site.D + h->site.n_neurons + 16);
  k_site_fp64<<<grid, 32 * SITE64_WARPS, smem, st>>>(
      h->d_sc, h->d_bm, h->site, h->at<int>(c.dense_list), n, c.npad, h->at<int4>(c.xyzt), h->at<int>(c.nl_r),
      h->at<unsigned long long>(c.amask), amask_words(h->p), h->at<int>(c.perm), pos, h->at<float>(c.q_radial), h->at<float>(c.u_site),
      h->at<AtomRec>(c.dk), h->at<float4>(c.pforce), want_q ? h->at<float>(c.q_desc) : nullptr);
}

// S3-S7 (+S5): outputs in the caller's order; any of energy/force/virial may be null.
template <class MS>
void enqueue_eval_t(nepzbl_handle* h, const double* pos, double* energy, float* force, float* virial,
                    bool want_q, bool with_zbl, const KickArgs& ka) {
  const Carve& c = h->cv;
  const int n = (int)h->n, npad = c.npad;
  cudaStream_t st = h->stream;
  const DenseArgs da{h->d_sc, h->dense_on ? h->at<int>(c.dense_list) : nullptr};
  const ModelTables<MS>& mt = *reinterpret_cast<const ModelTables<MS>*>(h->tables.data());
  const int gb = h->gather_block ? h->gather_block : ((long long)n * RADIAL_LANES < 8ll * 1024 * h->n_sm ? 32 : 64);
  prof_mark(h, PK_RADIAL);
  // cap_angular > 64: two mask words per atom (AW = 2 instantiations; the FFMA angular kernel, 64-thread k_force)
  const bool two_words = amask_words(h->p) > 1;
  auto launch_radial = [&](auto tri, auto stage, auto aw) {
    constexpr int STAGE = decltype(stage)::value;
    constexpr int AW = decltype(aw)::value;
    const int blk = STAGE ? STAGE_TILE * RADIAL_LANES : gb;
    const size_t smem = STAGE ? ((sizeof(TileDesc) + 8 + 15) / 16) * 16 + sizeof(int4) * STAGE_CAP : 0;
    if (STAGE) cudaFuncSetAttribute((const void*)k_radial<MS, decltype(tri)::value, STAGE, AW>,
                                    cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    k_radial<MS, decltype(tri)::value, STAGE, AW><<<blocks((long long)n * RADIAL_LANES, blk), blk, smem, st>>>(
        h->d_sc, h->d_bm, n, npad, h->at<int4>(c.xyzt), h->at<int>(c.nn_r), h->at<int>(c.nl_r), mt,
        h->at<float>(c.q_radial), h->at<unsigned>(c.rmask), h->at<unsigned>(c.tmask), mask_words(h->p), h->at<int>(c.zbl_list),
        h->at<int>(c.nn_a), h->at<unsigned long long>(c.amask), h->at<float4>(c.adisp),
        h->at<unsigned long long>(c.shellq), STAGE ? h->at<TileDesc>(c.tiles) : nullptr,
        STAGE ? h->at<unsigned short>(c.nl_loc) : nullptr);
  };
  using std::integral_constant;
  using one = integral_constant<int, 1>;
  using two = integral_constant<int, 2>;
  if (two_words && h->tri) launch_radial(std::true_type{}, integral_constant<int, 0>{}, two{});
  else if (two_words) launch_radial(std::false_type{}, integral_constant<int, 0>{}, two{});
  else if (h->tri) launch_radial(std::true_type{}, integral_constant<int, 0>{}, one{});
  else if (std::is_same<MS, MS0>::value && stage_mode() == 1) launch_radial(std::false_type{}, integral_constant<int, std::is_same<MS, MS0>::value ? 1 : 0>{}, one{});
  else if (std::is_same<MS, MS0>::value && stage_mode() == 2) launch_radial(std::false_type{}, integral_constant<int, std::is_same<MS, MS0>::value ? 2 : 0>{}, one{});
  else launch_radial(std::false_type{}, integral_constant<int, 0>{}, one{});
  prof_mark(h, PK_ANGULAR_NN);
  if constexpr (kSplit<MS>) {
    auto launch_split = [&](auto aw) {
      k_angular_nn_split<MS, decltype(aw)::value><<<std::min(blocks((long long)n * SPLIT_LANES, SPLIT_THREADS), h->ang_grid), SPLIT_THREADS, h->smem_nn, st>>>(
          n, npad, h->at<int4>(c.xyzt), h->at<unsigned long long>(c.amask), h->at<float4>(c.adisp), mt, h->d_nnw,
          h->at<float>(c.q_radial), h->at<float>(c.u_site), h->at<AtomRec>(c.dk), h->at<float4>(c.pforce),
          want_q ? h->at<float>(c.q_desc) : nullptr, da);
    };
    bool done = false;
    if constexpr (kSplitTc<MS>) {
      if (h->split_tc && !two_words) {
        k_angular_split_tc<MS><<<std::min(blocks(n, 128), h->ang_grid), STC_THREADS, h->smem_nn, st>>>(
            n, npad, h->at<int4>(c.xyzt), h->at<unsigned long long>(c.amask), h->at<float4>(c.adisp), mt, h->d_nnw,
            h->at<float>(c.q_radial), h->at<float>(c.u_site), h->at<AtomRec>(c.dk), h->at<float4>(c.pforce),
            want_q ? h->at<float>(c.q_desc) : nullptr, da);
        done = true;
      }
    }
    if (done) {}
    else if (two_words) launch_split(two{}); else launch_split(one{});
  } else {
    auto launch_nn = [&](auto mode, auto aw) {
      constexpr int NN = decltype(mode)::value;
      constexpr int TH = NN == 2 ? 128 : ANG_THREADS;
      k_angular_nn<MS, NN, decltype(aw)::value><<<std::min(blocks(n, TH), h->ang_grid), TH, h->smem_nn, st>>>(
          n, npad, h->at<int4>(c.xyzt), h->at<unsigned long long>(c.amask), h->at<float4>(c.adisp), mt, h->d_nnw,
          h->at<float>(c.q_radial), h->at<float>(c.u_site), h->at<AtomRec>(c.dk), h->at<float4>(c.pforce),
          want_q ? h->at<float>(c.q_desc) : nullptr, da);
    };
    if (two_words) launch_nn(std::integral_constant<int, 0>{}, two{});  // nn_mode is 0 (nep_zbl_create)
    else if (h->nn_mode == 3)
      k_angular_tc<MS><<<std::min(blocks(n, TCP_THREADS), h->ang_grid), TCP_THREADS, h->smem_nn, st>>>(
          n, npad, h->at<int4>(c.xyzt), h->at<unsigned long long>(c.amask), h->at<float4>(c.adisp), mt, h->d_nnw,
          h->at<float>(c.q_radial), h->at<float>(c.u_site), h->at<AtomRec>(c.dk), h->at<float4>(c.pforce),
          want_q ? h->at<float>(c.q_desc) : nullptr, da);
    else if (h->nn_mode == 2) launch_nn(std::integral_constant<int, 2>{}, one{});
    else if (h->nn_mode == 1) launch_nn(std::integral_constant<int, 1>{}, one{});
    else launch_nn(std::integral_constant<int, 0>{}, one{});
  }
  if (h->dense_on) {
    prof_mark(h, PK_SITE64);
    launch_site_fp64(h, pos, want_q, st);
    h->launches++;
  }
  prof_mark(h, PK_FORCE);
  auto launch_force_t = [&](auto vir, auto blk, auto tri, auto aw) {
    constexpr bool VIR = decltype(vir)::value;
    constexpr int BLK = decltype(blk)::value;
    k_force<MS, VIR, BLK, decltype(tri)::value, decltype(aw)::value><<<blocks((long long)n * FORCE_LANES, BLK), BLK, 0, st>>>(
        h->d_bm, n, npad, h->at<int4>(c.xyzt), h->at<int>(c.nn_r), h->at<int>(c.nl_r), h->at<int>(c.nn_a),
        h->at<int>(c.nl_r), h->at<unsigned char>(c.rev), mt, h->at<AtomRec>(c.dk), h->at<unsigned>(c.rmask),
        h->at<unsigned>(c.tmask), mask_words(h->p), h->at<unsigned long long>(c.amask), h->at<float4>(c.pforce), h->at<float>(c.u_site),
        h->at<int>(c.perm), energy, force, VIR ? virial : nullptr, ka);
  };
  // triclinic boxes take the 64-thread variant only (a NEXT row: fewer instantiations)
  auto launch_force = [&](auto vir, auto blk) {
    if (two_words && h->tri) launch_force_t(vir, std::integral_constant<int, 64>{}, std::true_type{}, two{});
    else if (two_words) launch_force_t(vir, std::integral_constant<int, 64>{}, std::false_type{}, two{});
    else if (h->tri) launch_force_t(vir, std::integral_constant<int, 64>{}, std::true_type{}, one{});
    else launch_force_t(vir, blk, std::false_type{}, one{});
  };
  if (virial) {
    if (gb == 32) launch_force(std::true_type{}, integral_constant<int, 32>{});
    else launch_force(std::true_type{}, integral_constant<int, 64>{});
  } else {
    if (gb == 32) launch_force(std::false_type{}, integral_constant<int, 32>{});
    else launch_force(std::false_type{}, integral_constant<int, 64>{});
  }
  h->launches += 3;
  if (h->p.zbl_enabled && with_zbl) {
    prof_mark(h, PK_ZBL);
    k_zbl<<<zbl_grid(h), 64, 0, st>>>(h->d_sc, h->d_bm, h->at<int>(c.zbl_list), n, npad, h->at<int4>(c.xyzt),
                            h->at<int>(c.nn_r), h->at<int>(c.nl_r), h->at<int>(c.perm), pos, h->zp,
                            energy, force, virial, ka);
    h->launches++;
  }
  prof_mark(h, -1);
}

void enqueue_eval(nepzbl_handle* h, const double* pos, double* energy, float* force, float* virial,
                  bool want_q, bool with_zbl = true, const KickArgs& ka = KickArgs{}) {
  with_shape(h->shape, [&](auto ms) { enqueue_eval_t<decltype(ms)>(h, pos, energy, force, virial, want_q, with_zbl, ka); });
}

void enqueue_zbl(nepzbl_handle* h, const double* pos, double* energy, float* force, float* virial, cudaStream_t st,
                 const KickArgs& ka) {
  const Carve& c = h->cv;
  k_zbl<<<zbl_grid(h), 64, 0, st>>>(h->d_sc, h->d_bm, h->at<int>(c.zbl_list), (int)h->n, c.npad, h->at<int4>(c.xyzt),
                          h->at<int>(c.nn_r), h->at<int>(c.nl_r), h->at<int>(c.perm), pos, h->zp, energy, force, virial, ka);
}

int read_scalars(nepzbl_handle* h) {
  CU(cudaMemcpyAsync(h->h_sc, h->d_sc, sizeof(Scalars), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  CU(cudaGetLastError());
  return NEPZBL_OK;
}

__global__ void k_clear_errors(Scalars* sc);
void destroy_step_graph(nepzbl_handle* h);

int check_device_flags(nepzbl_handle* h) {
  const Scalars& s = *h->h_sc;
  if (s.nonfinite || s.box_too_small || s.bad_type || s.overflow_radial > h->p.cap_radial ||
      s.overflow_angular > h->p.cap_angular) {  // errors are reported once, then cleared
    k_clear_errors<<<1, 1, 0, h->stream>>>(h->d_sc);
    h->launches++;
  }
  if (s.nonfinite) {
    h->have_list = false;
    return fail(h, NEPZBL_E_NONFINITE, "NaN/Inf in positions");
  }
  if (s.bad_type) {
    h->have_list = false;
    return fail(h, NEPZBL_E_INVALID_ARG, "an atom type is outside [0, n_types = %d)", h->p.n_types);
  }
  if (s.box_too_small) {
    h->have_list = false;
    return fail(h, NEPZBL_E_BOX_TOO_SMALL, "periodic box edge < 2*(rc_radial+skin)");
  }
  if (s.overflow_radial > h->p.cap_radial || s.overflow_angular > h->p.cap_angular) {
    h->have_list = false;
    return fail(h, NEPZBL_E_NEIGHBOR_OVERFLOW,
                "neighbour list overflow: an atom needs %d radial (cap %d) / %d angular (cap %d) slots",
                s.overflow_radial, h->p.cap_radial, s.overflow_angular, h->p.cap_angular);
  }
  return NEPZBL_OK;
}

int set_system(nepzbl_handle* h, long long n, const double box[9], const int32_t pbc[3], bool* changed) {
  if (!h->ws) return fail(h, NEPZBL_E_WORKSPACE, "no workspace set");
  if (n < 0 || n > h->n_cap) return fail(h, NEPZBL_E_WORKSPACE, "n = %lld exceeds workspace capacity %lld", n, h->n_cap);
  if (!box || !pbc) return fail(h, NEPZBL_E_INVALID_ARG, "box/pbc is NULL");
  bool tri = false;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b)
      if (a != b && box[3 * a + b] != 0.0) tri = true;
  double rcs = h->p.rc_radial + h->p.skin;
  double inv[9] = {0}, hgt[3] = {0};
  if (tri) {
    // triclinic (C-28): periodic along all three lattice vectors; every distance between opposite
    // faces must hold the minimum image
    if (!(pbc[0] && pbc[1] && pbc[2]))
      return fail(h, NEPZBL_E_BOX_NOT_ORTHOGONAL, "a non-orthogonal box must be periodic along all three lattice vectors");
    const double* H = box;
    const double c00 = H[4] * H[8] - H[5] * H[7], c01 = H[5] * H[6] - H[3] * H[8], c02 = H[3] * H[7] - H[4] * H[6];
    const double det = H[0] * c00 + H[1] * c01 + H[2] * c02;
    if (!(std::fabs(det) > 0.0) || !std::isfinite(det)) return fail(h, NEPZBL_E_INVALID_ARG, "box is singular");
    inv[0] = c00 / det; inv[1] = (H[2] * H[7] - H[1] * H[8]) / det; inv[2] = (H[1] * H[5] - H[2] * H[4]) / det;
    inv[3] = c01 / det; inv[4] = (H[0] * H[8] - H[2] * H[6]) / det; inv[5] = (H[2] * H[3] - H[0] * H[5]) / det;
    inv[6] = c02 / det; inv[7] = (H[1] * H[6] - H[0] * H[7]) / det; inv[8] = (H[0] * H[4] - H[1] * H[3]) / det;
    for (int a = 0; a < 3; ++a) {
      hgt[a] = 1.0 / std::sqrt(inv[a] * inv[a] + inv[3 + a] * inv[3 + a] + inv[6 + a] * inv[6 + a]);
      if (hgt[a] < 2.0 * rcs)
        return fail(h, NEPZBL_E_BOX_TOO_SMALL, "cell height %d = %g A < 2*(rc_radial+skin) = %g A", a, hgt[a], 2.0 * rcs);
    }
  } else {
    for (int a = 0; a < 3; ++a) {
      if (!(box[4 * a] > 0.0) || !std::isfinite(box[4 * a])) return fail(h, NEPZBL_E_INVALID_ARG, "box edge %d is not positive", a);
      if (pbc[a] && box[4 * a] < 2.0 * rcs)
        return fail(h, NEPZBL_E_BOX_TOO_SMALL, "periodic edge %d = %g A < 2*(rc_radial+skin) = %g A", a, box[4 * a], 2.0 * rcs);
    }
  }
  bool ch = !h->have_list || n != h->n;
  for (int a = 0; a < 9; ++a) ch = ch || box[a] != h->box[a];
  for (int a = 0; a < 3; ++a) ch = ch || (pbc[a] != 0) != (h->pbc[a] != 0);
  h->n = n;
  memcpy(h->box, box, sizeof h->box);
  for (int a = 0; a < 3; ++a) h->pbc[a] = pbc[a] != 0;
  h->tri = tri;
  memcpy(h->box_inv, inv, sizeof inv);
  memcpy(h->box_hgt, hgt, sizeof hgt);
  *changed = ch;
  return NEPZBL_OK;
}

void destroy_step_graph(nepzbl_handle* h) {
  if (h->step_exec) cudaGraphExecDestroy(h->step_exec);
  if (h->step_graph) cudaGraphDestroy(h->step_graph);
  h->step_exec = nullptr;
  h->step_graph = nullptr;
}

__global__ void k_set_force_rebuild(Scalars* sc) { sc->force_rebuild = 1; }

// FP32 FMA issue-rate microbenchmark: 16 independent register chains per thread (bench.py roofline peak)
__global__ void __launch_bounds__(512) k_ffma_peak(int iters, float m, float* sink) {
  float a[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = (float)(threadIdx.x + k) * 1e-3f;
  float b = m, c = 1e-7f * (float)blockIdx.x;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = fmaf(a[k], b, c);
  }
  float s = 0.0f;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k];
  if (s == 12345.678f) *sink = s;
}
__global__ void k_clear_errors(Scalars* sc) {
  sc->nonfinite = 0;
  sc->bad_type = 0;
  sc->box_too_small = 0;
  sc->overflow_radial = 0;
  sc->overflow_angular = 0;
}

int eval_common(nepzbl_handle* h, long long n, const double* pos, const int32_t* types,
                const double box[9], const int32_t pbc[3], double* energy, float* force, float* virial,
                bool force_rebuild, bool want_q, bool do_eval, bool from_md = false) {
  // A plain evaluation or list build on a handle with an MD session overwrites the lists, the sorted order and the
  // system size the session (and its captured graph) rely on: the session ends here, md_init starts a new one.
  if (!from_md && h->md_ready) {
    h->md_ready = false;
    destroy_step_graph(h);
  }
  bool changed = false;
  int rc = set_system(h, n, box, pbc, &changed);
  if (rc) return rc;
  if (n == 0) return NEPZBL_OK;
  if (!pos) return fail(h, NEPZBL_E_INVALID_ARG, "pos is NULL");
  const Carve& c = h->cv;
  const float skin = (float)h->p.skin;
  if (changed || force_rebuild) {
    k_set_force_rebuild<<<1, 1, 0, h->stream>>>(h->d_sc);
  } else {
    k_prep<<<blocks(n, 256), 256, 0, h->stream>>>(h->d_sc, h->d_bm, (int)n, pos, types, h->p.n_types,
                                                  h->at<int>(c.inv_perm), h->at<int4>(c.xyzt),
                                                  h->at<int4>(c.xyzt_build));
  }
  k_flag<<<1, 1, 0, h->stream>>>(h->d_sc, skin);
  h->launches += 2;
  prof_mark(h, PK_REBUILD);
  h->launches += enqueue_rebuild(h, pos, types, h->stream);
  if (do_eval) enqueue_eval(h, pos, energy, force, virial, want_q);
  rc = read_scalars(h);
  if (rc) return rc;
  rc = check_device_flags(h);
  if (rc) return rc;
  h->have_list = true;
  return NEPZBL_OK;
}

}  // namespace

// =============================================================================== C ABI

extern "C" {

int nep_zbl_create(const nepzbl_params* p, int device, void* cuda_stream, nepzbl_handle** out) {
  nepzbl_handle* h = nullptr;
  if (!p || !out) return fail(h, NEPZBL_E_INVALID_ARG, "params/out is NULL");
  *out = nullptr;
  if (p->n_types < 1 || p->n_types > 2) return fail(h, NEPZBL_E_UNSUPPORTED, "this build supports n_types 1 or 2 (got %d)", p->n_types);
  if (p->l_max != 4) return fail(h, NEPZBL_E_UNSUPPORTED, "this build supports l_max == 4 (got %d)", p->l_max);
  if (p->n_max_radial < 0 || p->n_max_angular < 0 || p->basis_radial < 0 || p->basis_angular < 0)
    return fail(h, NEPZBL_E_INVALID_ARG, "n_max / basis must be >= 0");
  // the instantiated shape this model runs on: an exact match, else the cheapest one that contains it (see kShapes)
  const ShapeId want{p->n_max_radial + 1, p->basis_radial + 1, p->n_max_angular + 1, p->basis_angular + 1,
                     p->has_4body != 0, p->n_types, p->has_5body != 0};
  auto fits = [&](const ShapeId& c) {
    return c.nr >= want.nr && c.kr >= want.kr && c.na >= want.na && c.ka >= want.ka && c.b4 >= want.b4 &&
           c.b5 >= want.b5 && c.nt == want.nt;
  };
  int shape = -1;
  for (int k = 0; k < (int)(sizeof kShapes / sizeof kShapes[0]); ++k) {
    const ShapeId& c = kShapes[k];
    if (c.nr == want.nr && c.kr == want.kr && c.na == want.na && c.ka == want.ka && c.b4 == want.b4 && c.b5 == want.b5 &&
        c.nt == want.nt)
      shape = k;
  }
  bool padded = false;
  if (shape < 0)
    for (int k : kShapeByCost)
      if (shape < 0 && fits(kShapes[k])) { shape = k; padded = true; }
  if (shape < 0)
    return fail(h, NEPZBL_E_UNSUPPORTED, "model shape n_max %d/%d basis %d/%d 4body %d 5body %d with %d atom type(s) fits no kernel of this build "
                "(n_max <= 15 / 10, basis <= 8; 5-body or 4-body with two types: n_max <= 4 / 4)",
                p->n_max_radial, p->n_max_angular, p->basis_radial, p->basis_angular, p->has_4body, p->has_5body, p->n_types);
  if (p->n_neurons < 1 || p->n_neurons > 256) return fail(h, NEPZBL_E_INVALID_ARG, "n_neurons out of range");
  if (p->cap_angular < 1 || p->cap_angular > 128 || p->cap_radial < 1 || p->cap_radial > 1024)
    return fail(h, NEPZBL_E_INVALID_ARG, "cap_angular must be in 1..128, cap_radial in 1..1024");
  if (!(p->rc_radial > 0) || !(p->rc_angular > 0) || p->rc_angular > p->rc_radial || p->skin < 0)
    return fail(h, NEPZBL_E_INVALID_ARG, "need 0 < rc_angular <= rc_radial and skin >= 0");
  if (p->zbl_enabled && (p->zbl_n_terms < 1 || p->zbl_n_terms > 4 || !(p->zbl_r_inner < p->zbl_r_outer) ||
                         p->zbl_r_outer + 0.01 > p->rc_radial))
    return fail(h, NEPZBL_E_INVALID_ARG, "bad ZBL parameters");
  if (!p->c_radial || !p->c_angular || !p->q_scaler || !p->w0 || !p->b0 || !p->w1 || !p->atomic_number || !p->mass)
    return fail(h, NEPZBL_E_INVALID_ARG, "a parameter array is NULL");

  // a model smaller than its kernel shape: zero-padded tables in the shape's sizes (its own descriptor components keep
  // their values; the padding channels have zero coefficients, hence zero components, and zero columns in w0)
  const int D_model = want.nr + 4 * want.na + (want.b4 ? want.na : 0) + (want.b5 ? want.na : 0);
  std::vector<int> qmap(D_model);       // descriptor component of the model -> component of the shape
  std::vector<double> pad_cr, pad_ca, pad_qs, pad_w0;
  nepzbl_params pp = *p;
  {
    const ShapeId& c = kShapes[shape];
    int v = 0;
    for (int n = 0; n < want.nr; ++n) qmap[v++] = desc_index(c.nr, c.na, c.b4, 0, n);
    for (int l = 1; l <= 4; ++l)
      for (int n = 0; n < want.na; ++n) qmap[v++] = desc_index(c.nr, c.na, c.b4, l, n);
    if (want.b4) for (int n = 0; n < want.na; ++n) qmap[v++] = desc_index(c.nr, c.na, c.b4, 5, n);
    if (want.b5) for (int n = 0; n < want.na; ++n) qmap[v++] = desc_index(c.nr, c.na, c.b4, 6, n);
    if (padded) {
      const int npr = c.nt * c.nt, Ds = c.nr + 4 * c.na + (c.b4 ? c.na : 0) + (c.b5 ? c.na : 0);
      pad_cr.assign((size_t)npr * c.nr * c.kr, 0.0);
      pad_ca.assign((size_t)npr * c.na * c.ka, 0.0);
      for (int pr = 0; pr < npr; ++pr) {
        for (int n = 0; n < want.nr; ++n)
          for (int k = 0; k < want.kr; ++k)
            pad_cr[((size_t)pr * c.nr + n) * c.kr + k] = p->c_radial[((size_t)pr * want.nr + n) * want.kr + k];
        for (int n = 0; n < want.na; ++n)
          for (int k = 0; k < want.ka; ++k)
            pad_ca[((size_t)pr * c.na + n) * c.ka + k] = p->c_angular[((size_t)pr * want.na + n) * want.ka + k];
      }
      pad_qs.assign(Ds, 0.0);
      pad_w0.assign((size_t)p->n_neurons * Ds, 0.0);
      for (int u = 0; u < D_model; ++u) {
        pad_qs[qmap[u]] = p->q_scaler[u];
        for (int m = 0; m < p->n_neurons; ++m) pad_w0[(size_t)m * Ds + qmap[u]] = p->w0[(size_t)m * D_model + u];
      }
      pp.n_max_radial = c.nr - 1; pp.basis_radial = c.kr - 1; pp.n_max_angular = c.na - 1; pp.basis_angular = c.ka - 1;
      pp.has_4body = c.b4; pp.has_5body = c.b5;
      pp.c_radial = pad_cr.data(); pp.c_angular = pad_ca.data(); pp.q_scaler = pad_qs.data(); pp.w0 = pad_w0.data();
      p = &pp;
    }
  }

  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev <= device || device < 0)
    return fail(h, NEPZBL_E_CUDA, "no CUDA device %d (%s): this library has no CPU fallback", device,
                e == cudaSuccess ? "device count too small" : cudaGetErrorString(e));
  h = new nepzbl_handle();
  h->p = *p;
  h->p.c_radial = h->p.c_angular = h->p.q_scaler = h->p.w0 = h->p.b0 = h->p.w1 = nullptr;
  h->p.atomic_number = h->p.mass = nullptr;
  h->shape = shape;
  h->device = device;
  h->stream = (cudaStream_t)cuda_stream;
  if (const char* ng = getenv("NEPZBL_NO_GRAPH")) h->use_graph = !(ng[0] == '1');  // see nepzbl.h (md_step)
  if (!h->use_graph) h->graph_note = "NEPZBL_NO_GRAPH=1";
  if (const char* gb = getenv("NEPZBL_GATHER_BLOCK")) {
    int v = atoi(gb);
    if (v == 32 || v == 64) h->gather_block = v;
  }
  if (amask_words(*p) > 1) h->nn_mode = 0;  // two mask words per atom: only the FFMA angular kernel is instantiated for them
  else if (const char* nm = getenv("NEPZBL_NN")) h->nn_mode = !strcmp(nm, "tc") ? 3 : (!strcmp(nm, "tcsync") ? 2 : (!strcmp(nm, "mma") ? 1 : 0));
  std::vector<float> nnw;
  with_shape(shape, [&](auto ms) {
    using MS = decltype(ms);
    build_tables<MS>(h, p);
    nnw = build_nnw<MS>(p);
    h->D = MS::D;
  });
  h->D_model = D_model;
  h->padded = padded;
  h->qmap = qmap;
  std::vector<double> site_tab;
  size_t site_off[6] = {0, 0, 0, 0, 0, 0};
  with_shape(shape, [&](auto ms) { site_tab = build_site_tables<decltype(ms)>(p, &h->site, site_off); });
  ZblParams& z = h->zp;
  memset(&z, 0, sizeof z);
  z.r_inner = p->zbl_r_inner; z.r_outer = p->zbl_r_outer; z.n_terms = p->zbl_n_terms;
  for (int k = 0; k < 4; ++k) { z.c[k] = p->zbl_c[k]; z.d[k] = p->zbl_d[k]; }
  z.a_num = p->zbl_a_num; z.a_pow = p->zbl_a_pow; z.coulomb_k = p->coulomb_k;
  for (int t = 0; t < p->n_types && t < 8; ++t) {
    z.Z[t] = p->atomic_number[t];
    z.Zpow[t] = pow(p->atomic_number[t], p->zbl_a_pow);
  }
  double zf = p->zbl_r_outer + 0.01;
  z.filter_r2 = (float)(zf * zf);

  auto die = [&](const char* what, cudaError_t ce) {
    std::string msg = std::string(what) + ": " + cudaGetErrorString(ce);
    nep_zbl_destroy(h);
    g_create_error = msg;
    return NEPZBL_E_CUDA;
  };
  cudaError_t ce;
  if ((ce = cudaSetDevice(device)) != cudaSuccess) return die("cudaSetDevice", ce);
  if (!h->stream) {
    // No stream given: the library makes its own BLOCKING stream.  It orders itself with the legacy default stream
    // (where a caller that passes NULL issues its own work) exactly as the default stream would, but -- unlike the
    // default stream -- it can be captured, so MD steps are replayed as a CUDA graph for such callers too.
    if ((ce = cudaStreamCreateWithFlags(&h->own_stream, cudaStreamDefault)) != cudaSuccess) return die("cudaStreamCreate", ce);
    h->stream = h->own_stream;
  }
  if ((ce = cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return die("cudaDeviceGetAttribute", ce);
  {  // k_angular_nn: opt in to its dynamic shared memory and size the persistent grid to the resident blocks
    const void* fn = nullptr;
    int threads = ANG_THREADS;
    with_shape(shape, [&](auto ms) {
      using MS = decltype(ms);
      if constexpr (kSplit<MS>) {
        fn = amask_words(*p) > 1 ? (const void*)k_angular_nn_split<MS, 2> : (const void*)k_angular_nn_split<MS, 1>;
        threads = SPLIT_THREADS;
        if constexpr (kSplitTc<MS>) {
          if (h->split_tc) { fn = (const void*)k_angular_split_tc<MS>; threads = STC_THREADS; }
        }
      }
      else if (amask_words(*p) > 1) fn = (const void*)k_angular_nn<MS, 0, 2>;
      else if (h->nn_mode == 3) { fn = (const void*)k_angular_tc<MS>; threads = TCP_THREADS; }
      else if (h->nn_mode == 2) { fn = (const void*)k_angular_nn<MS, 2>; threads = 128; }
      else fn = h->nn_mode == 1 ? (const void*)k_angular_nn<MS, 1> : (const void*)k_angular_nn<MS, 0>;
    });
    if ((ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_nn)) != cudaSuccess) return die("cudaFuncSetAttribute(k_angular_nn)", ce);
    // the tcgen05 variant needs two 105-KB blocks per SM: ask for the largest shared-memory carve-out
    if ((h->nn_mode >= 2 || h->split_tc) && (ce = cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)) != cudaSuccess)
      return die("cudaFuncSetAttribute(carveout)", ce);
    int per_sm = 0;
    if ((ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, h->smem_nn)) != cudaSuccess) return die("cudaOccupancyMaxActiveBlocksPerMultiprocessor", ce);
    if (per_sm < 1) return die("k_angular_nn does not fit one SM", cudaErrorInvalidConfiguration);
    // two blocks of the tcgen05 variant do fit an SM (2 x 128 x 256 registers, 2 x 105 KB: ncu's occupancy limits say 2 and
    // the measured kernel time halves against a one-block grid), but the occupancy query answers 1
    if (h->nn_mode >= 2 && per_sm < 2 && 2 * (h->smem_nn + 1024) <= 227 * 1024) per_sm = 2;
    if (const char* e = getenv("NEPZBL_ANG_BLOCKS_PER_SM")) {  // measurement aid: size of the persistent grid
      fprintf(stderr, "nepzbl: k_angular_nn occupancy %d block(s) of %d threads per SM, %zu bytes of shared memory\n", per_sm, threads, h->smem_nn);
      if (atoi(e) > 0) per_sm = atoi(e);
    }
    h->ang_grid = per_sm * h->n_sm;
  }
  if ((ce = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking)) != cudaSuccess) return die("cudaStreamCreate", ce);
  if ((ce = cudaEventCreateWithFlags(&h->ev_drift, cudaEventDisableTiming)) != cudaSuccess) return die("cudaEventCreate", ce);
  if ((ce = cudaMalloc(&h->d_sc, sizeof(Scalars))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMalloc(&h->d_bm, sizeof(BoxMap))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMalloc(&h->d_nnw, nnw.size() * sizeof(float))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMalloc(&h->d_qmap, h->qmap.size() * sizeof(int))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMalloc(&h->d_site, site_tab.size() * sizeof(double))) != cudaSuccess) return die("cudaMalloc", ce);
  h->site.ctA = h->d_site + site_off[0]; h->site.ctR = h->d_site + site_off[1]; h->site.qs = h->d_site + site_off[2];
  h->site.w0 = h->d_site + site_off[3]; h->site.b0 = h->d_site + site_off[4]; h->site.w1 = h->d_site + site_off[5];
  if ((ce = cudaMalloc(&h->d_mass, 8 * sizeof(double))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMalloc(&h->d_inv_mass, 8 * sizeof(double))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMalloc(&h->d_trace, kTraceRing * sizeof(double))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMalloc(&h->d_esum, 2 * sizeof(double))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMalloc(&h->d_nhc, sizeof(NhcState))) != cudaSuccess) return die("cudaMalloc", ce);
  if ((ce = cudaMallocHost(&h->h_nhc, sizeof(NhcState))) != cudaSuccess) return die("cudaMallocHost", ce);
  if ((ce = cudaMemsetAsync(h->d_nhc, 0, sizeof(NhcState), h->stream)) != cudaSuccess) return die("cudaMemset", ce);
  if ((ce = cudaMallocHost(&h->h_sc, sizeof(Scalars))) != cudaSuccess) return die("cudaMallocHost", ce);
  if ((ce = cudaMallocHost(&h->h_trace, kTraceRing * sizeof(double))) != cudaSuccess) return die("cudaMallocHost", ce);
  if ((ce = cudaMallocHost(&h->h_esum, 2 * sizeof(double))) != cudaSuccess) return die("cudaMallocHost", ce);
  double mass[8] = {0}, inv_mass[8] = {0};
  for (int t = 0; t < p->n_types && t < 8; ++t) {
    mass[t] = p->mass[t];
    inv_mass[t] = 1.0 / (p->mass[t] * NEPZBL_AMU_A2_FS2_TO_EV);
  }
  if ((ce = cudaMemsetAsync(h->d_sc, 0, sizeof(Scalars), h->stream)) != cudaSuccess) return die("cudaMemset", ce);
  if ((ce = cudaMemsetAsync(h->d_bm, 0, sizeof(BoxMap), h->stream)) != cudaSuccess) return die("cudaMemset", ce);
  if ((ce = cudaMemcpyAsync(h->d_nnw, nnw.data(), nnw.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream)) != cudaSuccess) return die("cudaMemcpy", ce);
  if ((ce = cudaMemcpyAsync(h->d_qmap, h->qmap.data(), h->qmap.size() * sizeof(int), cudaMemcpyHostToDevice, h->stream)) != cudaSuccess) return die("cudaMemcpy", ce);
  if ((ce = cudaMemcpyAsync(h->d_site, site_tab.data(), site_tab.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream)) != cudaSuccess) return die("cudaMemcpy", ce);
  if ((ce = cudaMemcpyAsync(h->d_mass, mass, sizeof mass, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess) return die("cudaMemcpy", ce);
  if ((ce = cudaMemcpyAsync(h->d_inv_mass, inv_mass, sizeof inv_mass, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess) return die("cudaMemcpy", ce);
  if ((ce = cudaStreamSynchronize(h->stream)) != cudaSuccess) return die("cudaStreamSynchronize", ce);
  *out = h;
  return NEPZBL_OK;
}

static void ws_free(nepzbl_handle* h) {
  auto& r = h->ws_ref;
  cudaFree(r.cell_of); cudaFree(r.cell_count); cudaFree(r.cell_fill); cudaFree(r.cell_start);
  cudaFree(r.occ); cudaFree(r.rec);
  r.cell_of = r.cell_count = r.cell_fill = r.cell_start = r.occ = nullptr;
  r.rec = nullptr;
  r.ns = 0;
}

void nep_zbl_destroy(nepzbl_handle* h) {
  if (!h) return;
  ws_free(h);
  cudaFree(h->ws_ref.out);
  cudaFreeHost(h->ws_ref.h_out);
  cudaFree(h->d_sc); cudaFree(h->d_bm); cudaFree(h->d_nnw); cudaFree(h->d_qmap); cudaFree(h->d_site); cudaFree(h->d_mass); cudaFree(h->d_inv_mass);
  cudaFree(h->d_trace); cudaFree(h->d_esum); cudaFree(h->d_nhc);
  cudaFreeHost(h->h_nhc);
  cudaFreeHost(h->h_sc); cudaFreeHost(h->h_trace); cudaFreeHost(h->h_esum);
  for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
  if (h->step_exec) cudaGraphExecDestroy(h->step_exec);
  if (h->step_graph) cudaGraphDestroy(h->step_graph);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  if (h->own_stream) cudaStreamDestroy(h->own_stream);
  if (h->ev_drift) cudaEventDestroy(h->ev_drift);
  delete h;
}

const char* nep_zbl_last_error(const nepzbl_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int nep_zbl_descriptor_dim(const nepzbl_handle* h) { return h ? h->D_model : 0; }

size_t nep_zbl_workspace_bytes(const nepzbl_handle* h, int64_t n_atoms) {
  if (!h || n_atoms < 0) return 0;
  return carve(h->p, h->D, n_atoms).total;
}

int nep_zbl_set_workspace(nepzbl_handle* h, void* dev_ptr, size_t bytes, int64_t n_atoms) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!dev_ptr || n_atoms < 0 || n_atoms > (1ll << 28)) return fail(h, NEPZBL_E_INVALID_ARG, "bad workspace arguments (n_atoms <= 2^28)");
  if (((uintptr_t)dev_ptr & 255) != 0) return fail(h, NEPZBL_E_WORKSPACE, "workspace must be 256-byte aligned");
  Carve c = carve(h->p, h->D, n_atoms);
  if (bytes < c.total) return fail(h, NEPZBL_E_WORKSPACE, "workspace too small: %zu < %zu bytes", bytes, c.total);
  h->ws = (char*)dev_ptr;
  h->ws_bytes = bytes;
  h->n_cap = n_atoms;
  h->cv = c;
  h->have_list = false;
  h->md_ready = false;
  return NEPZBL_OK;
}

int neighbor_build(nepzbl_handle* h, int64_t n, const double* pos, const int32_t* types,
                   const double box[9], const int32_t pbc[3]) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  return eval_common(h, n, pos, types, box, pbc, nullptr, nullptr, nullptr, true, false, false);
}

int neighbor_get(nepzbl_handle* h, int which, int32_t* nn, int32_t* nl) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->have_list) return fail(h, NEPZBL_E_STATE, "no neighbour list has been built");
  if (!nn || !nl || (which != 0 && which != 1)) return fail(h, NEPZBL_E_INVALID_ARG, "bad neighbor_get arguments");
  const Carve& c = h->cv;
  if (h->n > 0) {
    k_export_list<<<blocks(h->n, 128), 128, 0, h->stream>>>(
        (int)h->n, c.npad, which ? h->p.cap_angular : h->p.cap_radial, h->at<int>(c.perm),
        h->at<int>(which ? c.nn_a : c.nn_r), h->at<int>(c.nl_r), nn, nl);  // angular list = prefix
    h->launches++;
  }
  CU(cudaStreamSynchronize(h->stream));
  CU(cudaGetLastError());
  return NEPZBL_OK;
}

int nep_zbl_compute(nepzbl_handle* h, int64_t n, const double* pos, const int32_t* types,
                    const double box[9], const int32_t pbc[3], double* energy, float* force,
                    float* virial) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  return eval_common(h, n, pos, types, box, pbc, energy, force, virial, false, true, true);
}

int nep_zbl_compute_host(nepzbl_handle* h, int64_t n, const double* pos, const int32_t* types,
                         const double box[9], const int32_t pbc[3], double* energy, float* force,
                         float* virial) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->ws) return fail(h, NEPZBL_E_WORKSPACE, "no workspace set");
  if (n < 0 || n > h->n_cap) return fail(h, NEPZBL_E_WORKSPACE, "n exceeds workspace capacity");
  if (n == 0) return NEPZBL_OK;
  if (!pos) return fail(h, NEPZBL_E_INVALID_ARG, "pos is NULL");
  const Carve& c = h->cv;
  double* dpos = h->at<double>(c.st_pos);
  int32_t* dtyp = types ? h->at<int32_t>(c.st_types) : nullptr;
  CU(cudaMemcpyAsync(dpos, pos, 24 * (size_t)n, cudaMemcpyHostToDevice, h->stream));
  if (types) CU(cudaMemcpyAsync(dtyp, types, 4 * (size_t)n, cudaMemcpyHostToDevice, h->stream));
  double* de = energy ? h->at<double>(c.st_e) : nullptr;
  float* df = force ? h->at<float>(c.st_f) : nullptr;
  float* dw = virial ? h->at<float>(c.st_w) : nullptr;
  int rc = eval_common(h, n, dpos, dtyp, box, pbc, de, df, dw, false, true, true);
  if (rc) return rc;
  if (energy) CU(cudaMemcpyAsync(energy, de, 8 * (size_t)n, cudaMemcpyDeviceToHost, h->stream));
  if (force) CU(cudaMemcpyAsync(force, df, 12 * (size_t)n, cudaMemcpyDeviceToHost, h->stream));
  if (virial) CU(cudaMemcpyAsync(virial, dw, 36 * (size_t)n, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return NEPZBL_OK;
}

int nep_zbl_get_descriptors(nepzbl_handle* h, float* q) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->have_list) return fail(h, NEPZBL_E_STATE, "no evaluation has been made");
  if (!q) return fail(h, NEPZBL_E_INVALID_ARG, "q is NULL");
  const Carve& c = h->cv;
  if (h->n > 0) {
    k_export_q<<<blocks(h->n, 128), 128, 0, h->stream>>>((int)h->n, c.npad, h->D_model, h->d_qmap, h->at<int>(c.perm),
                                                        h->at<float>(c.q_desc), q);
    h->launches++;
  }
  CU(cudaStreamSynchronize(h->stream));
  CU(cudaGetLastError());
  return NEPZBL_OK;
}

// ---------------------------------------------------------------------------------- MD

static bool build_step_graph(nepzbl_handle* h);

int md_init(nepzbl_handle* h, int64_t n, double* pos, double* vel, const int32_t* types,
            const double box[9], const int32_t pbc[3]) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  h->md_ready = false;
  if (!pos || !vel) return fail(h, NEPZBL_E_INVALID_ARG, "pos/vel is NULL");
  bool changed;
  int rc = set_system(h, n, box, pbc, &changed);
  if (rc) return rc;
  if (n == 0) return fail(h, NEPZBL_E_INVALID_ARG, "md_init needs n > 0");
  const Carve& c = h->cv;
  CU(cudaMemsetAsync(h->d_sc, 0, sizeof(Scalars), h->stream));
  h->md_pos = pos;
  h->md_vel = vel;
  h->md_types = types;
  h->md_steps = 0;
  h->nhc_on = false;
  h->md_group = nullptr;
  rc = eval_common(h, n, pos, types, box, pbc, h->at<double>(c.md_energy), h->at<float>(c.md_force),
                   nullptr, true, false, true, true);
  if (rc) return rc;
  k_kick<<<blocks(n, 256), 256, 0, h->stream>>>(h->d_sc, (int)n, vel, h->at<float>(c.md_force), types,
                                                h->d_inv_mass, 0, 1);
  h->launches++;
  CU(cudaStreamSynchronize(h->stream));
  CU(cudaGetLastError());
  if (h->use_graph && !build_step_graph(h)) {  // falls back to plain stream launches; nep_zbl_uses_graph tells
    h->use_graph = false;
    h->graph_note = "CUDA graph capture of the MD step failed; steps are issued as plain stream launches";
  }
  h->md_ready = true;
  return NEPZBL_OK;
}

// one NHC(dt/2) operator on the thermostatted group (no-op unless md_set_thermostat
// enabled it).  phase 0: before the first half-kick (the scale factor is applied inside k_kick_drift);
// phase 1: after the second half-kick (k_scale_vmax applies it and leaves max |v|^2 for the next dt).
static int enqueue_nhc(nepzbl_handle* h, int phase, cudaStream_t st) {
  if (!h->nhc_on) return 0;
  const Carve& c = h->cv;
  const int n = (int)h->n;
  const int nb = (int)std::min<long long>(1024, (h->n + 255) / 256);
  k_group_ke2_partial<<<nb, 256, 0, st>>>(n, h->md_vel, h->md_types, h->d_mass, h->md_group,
                                          h->at<double>(c.nhc_partial), nullptr);
  k_nhc<<<1, 256, 0, st>>>(h->d_sc, h->d_nhc, nb, h->at<double>(c.nhc_partial), nullptr, phase);
  if (phase == 0) return 2;
  k_scale_vmax<<<blocks(n, 256), 256, 0, st>>>(h->d_sc, h->d_nhc, n, h->md_vel, h->md_group);
  return 3;
}

// One MD step as plain stream launches (profiling mode, or when graph capture is unavailable).
static void enqueue_md_step_stream(nepzbl_handle* h, bool trace) {
  const Carve& c = h->cv;
  const int n = (int)h->n;
  cudaStream_t st = h->stream;
  const float skin = (float)h->p.skin;
  prof_mark(h, PK_INTEGRATE_A);
  h->launches += enqueue_nhc(h, 0, st);
  k_kick_drift<<<blocks(n, 256), 256, 0, st>>>(h->d_sc, h->d_bm, n, h->md_pos, h->md_vel,
                                              h->at<float>(c.md_force), h->md_types, h->d_inv_mass,
                                              h->at<int>(c.inv_perm), h->at<int4>(c.xyzt),
                                              h->at<int4>(c.xyzt_build), h->nhc_on ? h->md_group : nullptr,
                                              h->d_nhc,
                                              StepFlagArgs{skin, trace ? h->d_trace : nullptr, kTraceRing, 0ull, 0, h->p.n_types});
  cudaEventRecord(h->ev_drift, st);
  h->launches += 1;
  prof_mark(h, PK_REBUILD);
  h->launches += enqueue_rebuild(h, h->md_pos, h->md_types, st);
  // S8b (second half-kick, max |v|^2) runs in the epilogue of k_force / in k_zbl
  enqueue_eval(h, h->md_pos, h->at<double>(c.md_energy), h->at<float>(c.md_force), nullptr, false, true,
               KickArgs{h->d_sc, h->md_vel, h->d_inv_mass, h->nhc_on ? 0 : 1, 0ull, 0});
  prof_mark(h, PK_KICK);
  h->launches += enqueue_nhc(h, 1, st);
  prof_mark(h, -1);
}


// Capture one MD step into a CUDA graph:
//   k_kick_drift (its last block: dt, rebuild decision) -> IF(rebuild){S2 chain} -> k_radial -> k_angular_nn
//   -> k_force (+ second half-kick, opens the ZBL node) -> IF(zbl_count > 0){k_zbl (+ kick of its atoms)}
//   5 kernels per step without rebuild / ZBL
// Returns false (and leaves the stream path in use) if any capture call fails.
static bool build_step_graph(nepzbl_handle* h) {
  destroy_step_graph(h);
  const Carve& c = h->cv;
  const int n = (int)h->n;
  cudaStream_t st = h->stream;
  const float skin = (float)h->p.skin;
  if (!h->cap_stream && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return false;
  cudaGraph_t g = nullptr;
  if (cudaGraphCreate(&g, 0) != cudaSuccess) return false;
  cudaGraphConditionalHandle h_reb, h_zbl;
  bool ok = cudaGraphConditionalHandleCreate(&h_reb, g, 0, cudaGraphCondAssignDefault) == cudaSuccess &&
            cudaGraphConditionalHandleCreate(&h_zbl, g, 0, cudaGraphCondAssignDefault) == cudaSuccess;
  ok = ok && cudaStreamBeginCaptureToGraph(st, g, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  if (!ok) { cudaGraphDestroy(g); cudaGetLastError(); return false; }
  bool saved_prof = h->prof;
  h->prof = false;
  long long saved_launches = h->launches;
  auto add_if = [&](cudaGraphConditionalHandle handle, cudaGraph_t* body) -> bool {
    cudaStreamCaptureStatus status;
    const cudaGraphNode_t* deps = nullptr;
    size_t ndeps = 0;
    cudaGraph_t cg = nullptr;
    if (cudaStreamGetCaptureInfo(st, &status, nullptr, &cg, &deps, &ndeps) != cudaSuccess) return false;
    cudaGraphNodeParams np = {};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = handle;
    np.conditional.type = cudaGraphCondTypeIf;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    if (cudaGraphAddNode(&node, g, deps, ndeps, &np) != cudaSuccess) return false;
    *body = np.conditional.phGraph_out[0];
    return cudaStreamUpdateCaptureDependencies(st, &node, 1, cudaStreamSetCaptureDependencies) == cudaSuccess;
  };
  int nk = 0, nk_reb = 0;
  nk += enqueue_nhc(h, 0, st);
  k_kick_drift<<<blocks(n, 256), 256, 0, st>>>(h->d_sc, h->d_bm, n, h->md_pos, h->md_vel,
                                              h->at<float>(c.md_force), h->md_types, h->d_inv_mass,
                                              h->at<int>(c.inv_perm), h->at<int4>(c.xyzt),
                                              h->at<int4>(c.xyzt_build), h->nhc_on ? h->md_group : nullptr,
                                              h->d_nhc,
                                              StepFlagArgs{skin, h->d_trace, kTraceRing, (unsigned long long)h_reb, 1, h->p.n_types});
  ok = ok && cudaEventRecordWithFlags(h->ev_drift, st, cudaEventRecordExternal) == cudaSuccess;
  nk += 1;
  cudaGraph_t body = nullptr;
  ok = ok && add_if(h_reb, &body);
  if (ok) {
    ok = cudaStreamBeginCaptureToGraph(h->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
      nk_reb = enqueue_rebuild(h, h->md_pos, h->md_types, h->cap_stream);
      ok = cudaStreamEndCapture(h->cap_stream, nullptr) == cudaSuccess;
    }
  }
  if (ok) {
    const KickArgs ka{h->d_sc, h->md_vel, h->d_inv_mass, h->nhc_on ? 0 : 1, (unsigned long long)h_zbl,
                      h->p.zbl_enabled ? 1 : 0};
    enqueue_eval(h, h->md_pos, h->at<double>(c.md_energy), h->at<float>(c.md_force), nullptr, false, false, ka);
    nk += 3 + (h->dense_on ? 1 : 0);
    if (h->p.zbl_enabled) {
      ok = add_if(h_zbl, &body);
      if (ok) {
        ok = cudaStreamBeginCaptureToGraph(h->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
        if (ok) {
          enqueue_zbl(h, h->md_pos, h->at<double>(c.md_energy), h->at<float>(c.md_force), nullptr, h->cap_stream, ka);
          ok = cudaStreamEndCapture(h->cap_stream, nullptr) == cudaSuccess;
        }
      }
    }
    nk += enqueue_nhc(h, 1, st);
  }
  cudaGraph_t captured = nullptr;
  cudaError_t ee = cudaStreamEndCapture(st, &captured);
  h->prof = saved_prof;
  h->launches = saved_launches;
  ok = ok && ee == cudaSuccess;
  if (ok) ok = cudaGraphInstantiate(&h->step_exec, g, 0) == cudaSuccess;
  if (!ok) {
    cudaGraphDestroy(g);
    h->step_exec = nullptr;
    cudaGetLastError();
    return false;
  }
  h->step_graph = g;
  h->graph_kernels = nk;
  h->graph_rebuild_kernels = nk_reb;
  return true;
}

// enqueue n_steps steps; dt_trace requests the device trace ring to be filled
static int enqueue_md_steps(nepzbl_handle* h, int n_steps, bool trace) {
  const bool graph = h->use_graph && !h->prof && h->step_exec;
  for (int k = 0; k < n_steps; ++k) {
    if (graph) {
      CU(cudaGraphLaunch(h->step_exec, h->stream));
      h->launches += h->graph_kernels;
    } else {
      enqueue_md_step_stream(h, trace);
    }
    h->md_steps++;
  }
  return NEPZBL_OK;
}

// one step; pos_host / vel_host (md_step_host): copy the new state out, the positions as soon as they are final
static int md_step_impl(nepzbl_handle* h, double dt_max, double max_displacement, double* dt_used, int32_t* rebuilt,
                        double* pos_host, double* vel_host) {
  if (!(dt_max > 0) || !(max_displacement > 0)) return fail(h, NEPZBL_E_INVALID_ARG, "dt_max and max_displacement must be > 0");
  k_md_params<<<1, 1, 0, h->stream>>>(h->d_sc, dt_max, max_displacement);
  h->launches++;
  int rc = enqueue_md_steps(h, 1, false);
  if (rc) return rc;
  if (pos_host) {
    const size_t b = 24 * (size_t)h->n;
    CU(cudaStreamWaitEvent(h->copy_stream, h->ev_drift, 0));
    CU(cudaMemcpyAsync(pos_host, h->md_pos, b, cudaMemcpyDeviceToHost, h->copy_stream));
    CU(cudaMemcpyAsync(vel_host, h->md_vel, b, cudaMemcpyDeviceToHost, h->stream));
  }
  rc = read_scalars(h);
  if (pos_host) {
    cudaError_t ce = cudaStreamSynchronize(h->copy_stream);
    if (!rc && ce != cudaSuccess) rc = fail(h, NEPZBL_E_CUDA, "copy stream: %s", cudaGetErrorString(ce));
  }
  if (rc) return rc;
  if (dt_used) *dt_used = h->h_sc->dt;
  if (rebuilt) *rebuilt = h->h_sc->do_rebuild;
  if (h->h_sc->do_rebuild && h->use_graph && !h->prof && h->step_exec) h->launches += h->graph_rebuild_kernels;
  if (h->h_sc->zbl_count > 0 && h->use_graph && !h->prof && h->step_exec) h->launches += 1;
  rc = check_device_flags(h);
  if (rc) h->md_ready = false;
  return rc;
}

int md_step(nepzbl_handle* h, double dt_max, double max_displacement, double* dt_used, int32_t* rebuilt) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready) return fail(h, NEPZBL_E_STATE, "md_step before md_init");
  return md_step_impl(h, dt_max, max_displacement, dt_used, rebuilt, nullptr, nullptr);
}

int md_run(nepzbl_handle* h, int64_t n_steps, double dt_max, double max_displacement, double* dt_trace,
           int64_t* n_rebuilds) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready) return fail(h, NEPZBL_E_STATE, "md_run before md_init");
  if (!(dt_max > 0) || !(max_displacement > 0) || n_steps < 0) return fail(h, NEPZBL_E_INVALID_ARG, "bad md_run arguments");
  int rc = read_scalars(h);
  if (rc) return rc;
  long long reb0 = h->h_sc->n_rebuilds;
  const bool graph = h->use_graph && !h->prof && h->step_exec;
  for (int64_t done = 0; done < n_steps;) {
    int chunk = (int)std::min<int64_t>(kTraceRing, n_steps - done);
    long long reb_before = h->h_sc->n_rebuilds;
    k_md_params<<<1, 1, 0, h->stream>>>(h->d_sc, dt_max, max_displacement);  // also rewinds the trace ring
    h->launches++;
    rc = enqueue_md_steps(h, chunk, true);
    if (rc) return rc;
    if (dt_trace) CU(cudaMemcpyAsync(h->h_trace, h->d_trace, chunk * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    rc = read_scalars(h);
    if (rc) return rc;
    if (dt_trace) memcpy(dt_trace + done, h->h_trace, chunk * sizeof(double));
    if (graph) h->launches += (h->h_sc->n_rebuilds - reb_before) * h->graph_rebuild_kernels;
    rc = check_device_flags(h);
    if (rc) { h->md_ready = false; return rc; }
    done += chunk;
  }
  if (n_rebuilds) *n_rebuilds = h->h_sc->n_rebuilds - reb0;
  return NEPZBL_OK;
}

int md_step_host(nepzbl_handle* h, double* pos, double* vel, double dt_max, double max_displacement,
                 double* dt_used, int32_t* rebuilt) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready) return fail(h, NEPZBL_E_STATE, "md_step_host before md_init");
  if (!pos || !vel) return fail(h, NEPZBL_E_INVALID_ARG, "pos/vel is NULL");
  size_t b = 24 * (size_t)h->n;
  CU(cudaMemcpyAsync(h->md_pos, pos, b, cudaMemcpyHostToDevice, h->stream));
  CU(cudaMemcpyAsync(h->md_vel, vel, b, cudaMemcpyHostToDevice, h->stream));
  return md_step_impl(h, dt_max, max_displacement, dt_used, rebuilt, pos, vel);
}

int md_request_rebuild(nepzbl_handle* h) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready) return fail(h, NEPZBL_E_STATE, "md_request_rebuild before md_init");
  k_set_force_rebuild<<<1, 1, 0, h->stream>>>(h->d_sc);
  h->launches++;
  CU(cudaGetLastError());
  return NEPZBL_OK;
}

int md_set_thermostat(nepzbl_handle* h, const uint8_t* group, double temperature, double tau,
                      int32_t chain_length) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready) return fail(h, NEPZBL_E_STATE, "md_set_thermostat before md_init");
  if (!group) {
    h->nhc_on = false;
    h->md_group = nullptr;
  } else {
    if (!(temperature > 0) || !(tau > 0) || chain_length < 1 || chain_length > NEPZBL_NHC_MAX)
      return fail(h, NEPZBL_E_INVALID_ARG, "need temperature > 0, tau > 0, 1 <= chain_length <= %d", NEPZBL_NHC_MAX);
    const Carve& c = h->cv;
    NhcState s;
    memset(&s, 0, sizeof s);
    s.enabled = 1;
    s.M = chain_length;
    s.kT = 8.617333262e-5 * temperature;
    s.tau = tau;
    s.scale = 1.0;
    *h->h_nhc = s;
    CU(cudaMemcpyAsync(h->d_nhc, h->h_nhc, sizeof s, cudaMemcpyHostToDevice, h->stream));
    const int nb = (int)std::min<long long>(1024, (h->n + 255) / 256);
    k_group_ke2_partial<<<nb, 256, 0, h->stream>>>((int)h->n, h->md_vel, h->md_types, h->d_mass, group,
                                                   h->at<double>(c.nhc_partial), h->at<double>(c.nhc_partial) + 1024);
    k_nhc<<<1, 256, 0, h->stream>>>(h->d_sc, h->d_nhc, nb, h->at<double>(c.nhc_partial),
                                    h->at<double>(c.nhc_partial) + 1024, 0);
    h->launches += 2;
    CU(cudaStreamSynchronize(h->stream));
    CU(cudaGetLastError());
    h->md_group = group;
    h->nhc_on = true;
  }
  if (h->use_graph && !build_step_graph(h)) {
    h->use_graph = false;
    h->graph_note = "CUDA graph capture of the thermostatted MD step failed; steps are issued as plain stream launches";
  }
  return NEPZBL_OK;
}

int md_set_thermostat_state(nepzbl_handle* h, const double* xi, const double* vxi) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready || !h->nhc_on) return fail(h, NEPZBL_E_STATE, "no thermostat is set");
  if (!xi || !vxi) return fail(h, NEPZBL_E_INVALID_ARG, "xi/vxi is NULL");
  CU(cudaMemcpyAsync(h->h_nhc, h->d_nhc, sizeof(NhcState), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  for (int k = 0; k < h->h_nhc->M; ++k) {
    h->h_nhc->xi[k] = xi[k];
    h->h_nhc->vxi[k] = vxi[k];
  }
  CU(cudaMemcpyAsync(h->d_nhc, h->h_nhc, sizeof(NhcState), cudaMemcpyHostToDevice, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return NEPZBL_OK;
}

int md_get_thermostat(nepzbl_handle* h, double* xi, double* vxi, double* t_group, double* conserved_extra) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready || !h->nhc_on) return fail(h, NEPZBL_E_STATE, "no thermostat is set");
  const Carve& c = h->cv;
  const int nb = (int)std::min<long long>(1024, (h->n + 255) / 256);
  k_group_ke2_partial<<<nb, 256, 0, h->stream>>>((int)h->n, h->md_vel, h->md_types, h->d_mass, h->md_group,
                                                 h->at<double>(c.nhc_partial), nullptr);
  k_energy_final<<<1, 256, 0, h->stream>>>(-nb, h->at<double>(c.nhc_partial), h->d_esum);
  h->launches += 2;
  CU(cudaMemcpyAsync(h->h_esum, h->d_esum, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaMemcpyAsync(h->h_nhc, h->d_nhc, sizeof(NhcState), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  CU(cudaGetLastError());
  const NhcState& s = *h->h_nhc;
  for (int k = 0; k < s.M; ++k) {
    if (xi) xi[k] = s.xi[k];
    if (vxi) vxi[k] = s.vxi[k];
  }
  if (t_group) *t_group = s.nf > 0 ? h->h_esum[0] / (s.nf * 8.617333262e-5) : 0.0;
  if (conserved_extra) {  // H' - E_kin - E_pot of ref. [32]
    double e = 0.0;
    for (int k = 0; k < s.M; ++k) {
      double w = (k == 0 ? s.nf : 1.0) * s.kT;
      e += 0.5 * w * s.tau * s.tau * s.vxi[k] * s.vxi[k] + w * s.xi[k];
    }
    *conserved_extra = e;
  }
  return NEPZBL_OK;
}

// ------------------------------------------------------------------ Wigner-Seitz count

int wigner_seitz_set_reference(nepzbl_handle* h, int64_t n_sites, const double* site_soa, const double box[9],
                               const int32_t pbc[3]) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (n_sites < 1 || n_sites > 2000000000ll || !site_soa || !box || !pbc)
    return fail(h, NEPZBL_E_INVALID_ARG, "bad wigner_seitz_set_reference arguments");
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b)
      if (a != b && box[3 * a + b] != 0.0)
        return fail(h, NEPZBL_E_BOX_NOT_ORTHOGONAL, "only orthogonal boxes are supported");
  for (int a = 0; a < 3; ++a)
    if (!(box[4 * a] > 0.0) || !std::isfinite(box[4 * a])) return fail(h, NEPZBL_E_INVALID_ARG, "box edge %d is not positive", a);
  auto& r = h->ws_ref;
  ws_free(h);
  const int ns = (int)n_sites;
  cudaStream_t st = h->stream;
  if (!r.out) CU(cudaMalloc(&r.out, 8 * sizeof(unsigned long long)));
  if (!r.h_out) CU(cudaMallocHost(&r.h_out, 8 * sizeof(unsigned long long)));
  // bounds of the sites (grid extent on open axes)
  for (int a = 0; a < 3; ++a) { r.h_out[a] = ~0ull; r.h_out[3 + a] = 0ull; }
  CU(cudaMemcpyAsync(r.out, r.h_out, 6 * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
  k_ws_bounds<<<blocks(ns, 256), 256, 0, st>>>(ns, site_soa, r.out);
  CU(cudaMemcpyAsync(r.h_out, r.out, 6 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  h->launches += 1;
  WsGrid g;
  memset(&g, 0, sizeof g);
  double ext[3], vol = 1.0;
  for (int a = 0; a < 3; ++a) {
    g.pbc[a] = pbc[a] != 0;
    g.L[a] = box[4 * a];
    if (g.pbc[a]) {
      g.lo[a] = 0.0;
      ext[a] = box[4 * a];
    } else {
      auto dec = [](unsigned long long k) {
        unsigned long long b = (k & 0x8000000000000000ull) ? (k & 0x7fffffffffffffffull) : ~k;
        double x;
        memcpy(&x, &b, 8);
        return x;
      };
      double mn = dec(r.h_out[a]), mx = dec(r.h_out[3 + a]);
      if (!(mx >= mn)) return fail(h, NEPZBL_E_NONFINITE, "no finite reference site coordinates");
      g.lo[a] = mn;
      ext[a] = std::max(mx - mn, 1e-9);
    }
    vol *= ext[a];
  }
  // cells of about 4 sites: edge = cbrt(4 V / n_sites) (bcc W: 1.26 a0 = 4 A, well above the ~1.5 A an atom of
  // a crystal sits from its nearest site, so the 27-cell block settles it)
  const double edge = cbrt(4.0 * vol / (double)ns);
  long long total = 1;
  for (int a = 0; a < 3; ++a) {
    long long nc = (long long)floor(ext[a] / edge);
    if (nc < 1) nc = 1;
    if (nc > 2048) nc = 2048;
    g.nc[a] = (int)nc;
    g.w[a] = ext[a] / (double)nc;
    g.inv_w[a] = (double)nc / ext[a];
    total *= nc;
  }
  // never more cells than sites: a degenerate extent (all sites in one plane of an open axis, a single site) makes
  // `edge` tiny, and a grid of millions of empty cells turns the ring-by-ring search of an atom far from every site
  // into minutes (found by tests/test_gpu_ws.py::test_degenerate_inputs: 88 s for ONE site); also keeps ints safe
  while (total > std::max<long long>(1, std::min<long long>(ns, 2000000000ll))) {
    int a = g.nc[0] >= g.nc[1] && g.nc[0] >= g.nc[2] ? 0 : (g.nc[1] >= g.nc[2] ? 1 : 2);
    total /= g.nc[a];
    g.nc[a] = (g.nc[a] + 1) / 2;
    g.w[a] = ext[a] / g.nc[a];
    g.inv_w[a] = g.nc[a] / ext[a];
    total *= g.nc[a];
  }
  g.ncells = (int)total;
  CU(cudaMalloc(&r.cell_of, sizeof(int) * (size_t)ns));
  CU(cudaMalloc(&r.cell_count, sizeof(int) * ((size_t)g.ncells + 1)));
  CU(cudaMalloc(&r.cell_fill, sizeof(int) * ((size_t)g.ncells + 1)));
  CU(cudaMalloc(&r.cell_start, sizeof(int) * ((size_t)g.ncells + 1)));
  CU(cudaMalloc(&r.occ, sizeof(int) * (size_t)ns));
  CU(cudaMalloc(&r.rec, sizeof(WsSite) * (size_t)ns));
  CU(cudaMemsetAsync(r.cell_count, 0, sizeof(int) * ((size_t)g.ncells + 1), st));
  CU(cudaMemsetAsync(r.cell_fill, 0, sizeof(int) * ((size_t)g.ncells + 1), st));
  k_ws_bin<<<blocks(ns, 256), 256, 0, st>>>(g, ns, site_soa, r.cell_of, r.cell_count);
  k_ws_scan<<<1, 1024, 0, st>>>(g.ncells, r.cell_count, r.cell_start);
  k_ws_place<<<blocks(ns, 256), 256, 0, st>>>(ns, site_soa, r.cell_of, r.cell_start, r.cell_fill, r.rec);
  h->launches += 3;
  CU(cudaStreamSynchronize(st));
  CU(cudaGetLastError());
  r.g = g;
  r.ns = ns;
  return NEPZBL_OK;
}

int wigner_seitz_count(nepzbl_handle* h, int64_t n, const double* pos_soa, int32_t* nearest, int32_t* occupancy,
                       int64_t* n_vacancies, int64_t* n_interstitials) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  auto& r = h->ws_ref;
  if (r.ns < 1) return fail(h, NEPZBL_E_STATE, "wigner_seitz_count before wigner_seitz_set_reference");
  if (n < 0 || n > 2000000000ll || (n > 0 && !pos_soa)) return fail(h, NEPZBL_E_INVALID_ARG, "bad wigner_seitz_count arguments");
  cudaStream_t st = h->stream;
  int* occ = occupancy ? occupancy : r.occ;
  CU(cudaMemsetAsync(occ, 0, sizeof(int) * (size_t)r.ns, st));
  CU(cudaMemsetAsync(r.out, 0, 2 * sizeof(unsigned long long), st));
  if (n > 0) {
    k_ws_assign<<<blocks(n, 128), 128, 0, st>>>(r.g, (int)n, pos_soa, r.cell_start, r.rec, nearest, occ);
    h->launches += 1;
  }
  k_ws_count<<<std::min(blocks(r.ns, 256), 1184), 256, 0, st>>>((int)r.ns, occ, r.out);
  h->launches += 1;
  CU(cudaMemcpyAsync(r.h_out, r.out, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  CU(cudaGetLastError());
  if (n_vacancies) *n_vacancies = (int64_t)r.h_out[0];
  if (n_interstitials) *n_interstitials = (int64_t)r.h_out[1];
  return NEPZBL_OK;
}

int md_energies(nepzbl_handle* h, double* e_pot, double* e_kin) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready) return fail(h, NEPZBL_E_STATE, "md_energies before md_init");
  const Carve& c = h->cv;
  int nb = (int)std::min<long long>(1024, (h->n + 255) / 256);
  k_energy_partial<<<nb, 256, 0, h->stream>>>((int)h->n, h->md_vel, h->at<double>(c.md_energy), h->md_types,
                                              h->d_mass, h->at<double>(c.partial));
  k_energy_final<<<1, 256, 0, h->stream>>>(nb, h->at<double>(c.partial), h->d_esum);
  h->launches += 2;
  CU(cudaMemcpyAsync(h->h_esum, h->d_esum, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  CU(cudaGetLastError());
  if (e_pot) *e_pot = h->h_esum[0];
  if (e_kin) *e_kin = h->h_esum[1];
  return NEPZBL_OK;
}

int md_get_forces(nepzbl_handle* h, float* force, double* energy) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready) return fail(h, NEPZBL_E_STATE, "md_get_forces before md_init");
  const Carve& c = h->cv;
  if (force) CU(cudaMemcpyAsync(force, h->at<float>(c.md_force), 12 * (size_t)h->n, cudaMemcpyDeviceToDevice, h->stream));
  if (energy) CU(cudaMemcpyAsync(energy, h->at<double>(c.md_energy), 8 * (size_t)h->n, cudaMemcpyDeviceToDevice, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return NEPZBL_OK;
}

int md_get_counters(nepzbl_handle* h, int64_t* n_steps, int64_t* n_rebuilds, int64_t* n_zbl_atoms) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->md_ready) return fail(h, NEPZBL_E_STATE, "md_get_counters before md_init");
  int rc = read_scalars(h);
  if (rc) return rc;
  if (n_steps) *n_steps = h->h_sc->n_steps;
  if (n_rebuilds) *n_rebuilds = h->h_sc->n_rebuilds;
  if (n_zbl_atoms) *n_zbl_atoms = h->h_sc->zbl_count;
  return NEPZBL_OK;
}

int nep_zbl_network_mode(const nepzbl_handle* h) {
  if (!h) return -1;
  bool split = false;
  with_shape(h->shape, [&](auto ms) { split = kSplit<decltype(ms)>; });
  return split ? (h->split_tc ? 3 : 0) : h->nn_mode;
}

int nep_zbl_uses_graph(const nepzbl_handle* h) {
  return h && h->md_ready && h->use_graph && h->step_exec ? 1 : 0;
}

int nep_zbl_last_counts(nepzbl_handle* h, int64_t* n_zbl_atoms, int64_t* n_fp64_atoms) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  if (!h->have_list) return fail(h, NEPZBL_E_STATE, "no evaluation has been made");
  int rc = read_scalars(h);
  if (rc) return rc;
  if (n_zbl_atoms) *n_zbl_atoms = h->h_sc->zbl_count;
  if (n_fp64_atoms) *n_fp64_atoms = h->h_sc->dense_count;
  return NEPZBL_OK;
}

int64_t nep_zbl_launch_count(const nepzbl_handle* h) { return h ? h->launches : 0; }

int nep_zbl_profile(nepzbl_handle* h, int enable) {
  if (!h) return NEPZBL_E_INVALID_ARG;
  CU(cudaStreamSynchronize(h->stream));
  h->prof = enable != 0;
  h->spans.clear();
  h->ev_used = 0;
  h->ev_open_id = -1;
  return NEPZBL_OK;
}

int nep_zbl_profile_read(nepzbl_handle* h, double* ms, int64_t* counts) {
  if (!h || !ms || !counts) return NEPZBL_E_INVALID_ARG;
  CU(cudaStreamSynchronize(h->stream));
  for (int k = 0; k < NEPZBL_PROFILE_SLOTS; ++k) { ms[k] = 0.0; counts[k] = 0; }
  for (const auto& sp : h->spans) {
    float t = 0.0f;
    CU(cudaEventElapsedTime(&t, sp.a, sp.b));
    if (sp.id >= 0 && sp.id < NEPZBL_PROFILE_SLOTS) { ms[sp.id] += t; counts[sp.id] += 1; }
  }
  h->spans.clear();
  h->ev_used = 0;
  h->ev_open_id = -1;
  return NEPZBL_OK;
}

int nep_zbl_ffma_peak(nepzbl_handle* h, double* tflops) {
  if (!h || !tflops) return NEPZBL_E_INVALID_ARG;
  int sms = 0;
  CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device));
  float* sink = nullptr;
  CU(cudaMalloc(&sink, sizeof(float)));
  cudaEvent_t a, b;
  CU(cudaEventCreate(&a));
  CU(cudaEventCreate(&b));
  const int iters = 4096, grid = sms * 8, block = 512;
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    CU(cudaEventRecord(a, h->stream));
    k_ffma_peak<<<grid, block, 0, h->stream>>>(iters, 1.0001f, sink);
    CU(cudaEventRecord(b, h->stream));
    CU(cudaEventSynchronize(b));
    float t = 0.0f;
    CU(cudaEventElapsedTime(&t, a, b));
    double fl = 2.0 * 16.0 * iters * (double)grid * block;  // 16 independent FMA chains per thread
    if (rep > 0) best = std::max(best, fl / (t * 1e-3) * 1e-12);
  }
  h->launches += 5;
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(sink);
  *tflops = best;
  return NEPZBL_OK;
}

}  // extern "C"
