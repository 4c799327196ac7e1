// clip.cu -- host side of libclip: the C ABI of include/clip.h.  No device allocation happens here: the caller's
// workspace is carved into the arrays listed at the top of clip_kernels.cuh.
#include "../../include/clip.h"
#include "clip_kernels.cuh"
#include "clip_fast.cuh"
#include "clip_fused.cuh"
#include "clip_d2q9.cuh"
#include "clip_launch.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

namespace {

char g_create_error[256] = "";

void set_err(char* dst, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 256, fmt, ap);
  va_end(ap);
}

constexpr size_t ALIGN = 256;
size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
  size_t word;  // 4 or 8
  size_t off_p[2], off_phi, off_u, off_obf, off_obg, off_lam, off_mask, off_phi2, off_part, total;
};

// Tiling of the single-pass kernel k_fused (clip_fused.cuh): tiles of `ty` rows x one z chunk; the number of tiles is
// chosen close to (and not above) a whole number of waves of resident blocks on the 148 SMs of a B200.
struct FusedPlan {
  bool ok, fills_gpu, pays, tma, tma_g;  // tma: path 4, k_fused_tma (bulk-async feed) admitted
  int ty, ytiles, nchunks, tzmax, threads, blocks_per_sm;
  int cs;  // y-adjacent tiles per thread-block cluster (1: none): k_fused<..., CL = true>
  int zc[clip::FUSED_MAX_CHUNKS + 1];  // chunk boundaries along z
  size_t part_words, smem_bytes;
};
constexpr int B200_SMS = 148;


FusedPlan fused_plan(int nx, int ny, int nz, const clip_params* p) {
  FusedPlan f{};
  if (p->collision != CLIP_COLL_WMRT || p->phase_only || p->lattice != 0) return f;
  for (int k = 0; k < 4; ++k) if (p->bc[k] != CLIP_BC_PERIODIC && p->bc[k] != CLIP_BC_WALL && p->bc[k] != CLIP_BC_FREESLIP) return f;
  if (p->bc[4] == CLIP_BC_FREESLIP || p->bc[5] == CLIP_BC_FREESLIP) return f;
  // an INLET / OUTLET plane is stepped by the generic kernels, the ghost plane of a HALO face not at all; k_fused covers the
  // planes [zlo, zlo + nz) in between
  const int zlo = (p->bc[4] == CLIP_BC_INLET || p->bc[4] == CLIP_BC_HALO) ? 1 : 0;
  nz -= zlo + ((p->bc[5] == CLIP_BC_OUTLET || p->bc[5] == CLIP_BC_HALO) ? 1 : 0);
  if (nx % 64 != 0 || nx > 512 || ny % 4 != 0 || nz < 4) return f;
  f.ty = 4;  // small tiles leave more of the SM's L1 to the phi stencil and the shifted population loads (measured)
  if ((p->tile_ty == 4 || p->tile_ty == 8 || p->tile_ty == 16) && ny % p->tile_ty == 0) f.ty = p->tile_ty;
  f.ytiles = ny / f.ty;
  f.threads = nx / 2;
  const int word = p->precision == 32 ? 4 : 8;
  const int nwarps = f.threads / 32;
  f.smem_bytes = (size_t)clip::FUSED_SLOTS * (f.ty + 2) * (nx + 2 * nwarps) * word;
  int bps = clip::fused_threads_per_sm(p->precision, f.threads) / f.threads;
  if (p->path == 4 || p->path == 5) {  // k_fused_tma: two stages of 38 (path 5, hybrid: 19) rows behind the ring; periodic x / y faces only
    bool periodic_xy = true;
    for (int k = 0; k < 4; ++k) periodic_xy = periodic_xy && p->bc[k] == CLIP_BC_PERIODIC;
    periodic_xy = periodic_xy && p->bc[4] != CLIP_BC_WALL && p->bc[5] != CLIP_BC_WALL;   // a z wall needs the wall body
    const size_t need = (f.smem_bytes + 127) / 128 * 128 + (size_t)clip::TMA_STAGES * (p->path == 5 ? 19 : 38) * nx * word + 64;
    if (periodic_xy && need + 1024 <= 227 * 1024) {
      f.tma = true; f.tma_g = p->path == 5; f.smem_bytes = need;
      const int by_smem = (int)((227 * 1024) / (need + 1024));
      bps = f.tma_g ? (bps < by_smem ? bps : by_smem) : by_smem;
    }
  }
  if (bps > 32) bps = 32;
  if (bps < 1) bps = 1;
  while (bps > 1 && (f.smem_bytes + 1024) * bps > 227 * 1024) --bps;
  if (f.smem_bytes + 1024 > 227 * 1024) return f;
  f.blocks_per_sm = bps;
  const long long cap = (long long)B200_SMS * bps;
  const int max_chunks = nz / 4 > 0 ? nz / 4 : 1;
  f.fills_gpu = (long long)f.ytiles * max_chunks >= cap;
  // measured: +4 .. +11 % at nx >= 256; at nx = 128 only with many waves of tiles (RT 128x512x128: +1 % fp32, +6 % fp64; 128^3: slower)
  f.pays = (nx >= 256 && f.fills_gpu) || (nx >= 128 && (long long)f.ytiles * max_chunks >= 4 * cap);
  // Chunks along z, dispatched in order (blockIdx.y): long ones (<= 16 planes: little halo traffic) first, then about one
  // wave of 8-plane and one wave of 4-plane chunks, so that the last blocks to finish are short ones (uniform chunks leave
  // ~4 % of the SM time idle in the last wave).  Small lattices and tile_chunks = n (tests) take n equal chunks.  The chunk
  // COUNT is bounded before anything is written to zc (FUSED_MAX_CHUNKS entries): long thin lattices get longer chunks.
  const int maxc = clip::FUSED_MAX_CHUNKS < nz ? clip::FUSED_MAX_CHUNKS : nz;
  int nchunks = 0, uniform = 0;
  if (p->tile_chunks >= 1) uniform = p->tile_chunks < maxc ? p->tile_chunks : maxc;
  const long long per_wave_ll = (cap + f.ytiles - 1) / f.ytiles;  // chunks that are resident at the same time
  const int per_wave = per_wave_ll > nz ? nz : (int)per_wave_ll;
  bool graded = !uniform && 12LL * per_wave <= nz / 2;
  if (graded) {
    const int rest = nz - 12 * per_wave, nl = (rest + 15) / 16;
    if ((long long)nl + 2LL * per_wave > maxc) graded = false;
    else {
      int z = 0;
      for (int k = 0; k < nl; ++k) { f.zc[nchunks++] = z; z += rest / nl + (k < rest % nl ? 1 : 0); }
      for (int k = 0; k < per_wave; ++k) { f.zc[nchunks++] = z; z += 8; }
      for (int k = 0; k < per_wave; ++k) { f.zc[nchunks++] = z; z += 4; }
      f.zc[nchunks] = nz;
    }
  }
  if (!graded) {
    if (!uniform) {  // as many equal chunks as fill a whole number of waves, at most 16 planes each (more where the count is bounded)
      for (int m = 1; m <= 64; ++m) {
        long long c = m * cap / f.ytiles;
        if (c < 1) continue;
        if (c > max_chunks) { if (uniform == 0) uniform = max_chunks; break; }
        uniform = (int)c;
        if ((nz + uniform - 1) / uniform <= 16) break;
      }
      if (uniform < 1) uniform = 1;
      if (uniform > maxc) uniform = maxc;
    }
    nchunks = uniform;
    for (int c = 0; c <= nchunks; ++c) f.zc[c] = (int)((long long)c * nz / nchunks);
  }
  for (int c = 0; c <= nchunks; ++c) f.zc[c] += zlo;
  f.nchunks = nchunks;
  f.tzmax = 1;
  for (int c = 0; c < nchunks; ++c) f.tzmax = f.zc[c + 1] - f.zc[c] > f.tzmax ? f.zc[c + 1] - f.zc[c] : f.tzmax;
  f.part_words = (size_t)f.ytiles * nchunks * (2 * f.tzmax + 2 * (f.ty + 2)) * nx;
  // Clusters of y-adjacent tiles (clip_fused.cuh, flush_slot_cl): measured to pay with the small blocks of nx = 128 (RT 128 x 512 x 128
  // fp32: +2.4 % with 4 tiles) and nx = 192 (the jets, fp32: +1 .. 2 % with 2); slower at nx >= 256 and in fp64 (the per-plane
  // barrier of the cluster couples the blocks; profiles/r02_experiments.md 4e)
  f.cs = p->cluster_y;
  if (f.cs == 0)   // ... and only with several waves of tiles (128^3 with k_fused forced: 0.166 against 0.139 ms)
    f.cs = (p->precision == 32 && !f.tma && (long long)f.ytiles * max_chunks >= 4 * cap) ? (nx == 128 ? 4 : (nx == 192 ? 2 : 1)) : 1;
  if (f.cs < 1 || f.tma || f.ytiles % f.cs != 0) f.cs = 1;
  f.ok = true;
  return f;
}

// Single-pass path of the D2Q9 lattice (clip_d2q9.cuh, k_fused9 + k_fix9): chunks of whole rows, one block each; as many chunks as
// fill a whole number of waves of resident blocks with at most 16 rows each.
struct Fused9Plan {
  bool ok, pays;
  int nchunks, threads;
  size_t smem_bytes, part_words;
};
Fused9Plan fused9_plan(int nx, int ny, const clip_params* p) {
  Fused9Plan f{};
  if (p->lattice != 1 || p->phase_only || nx % 64 != 0 || ny < 4 || p->path < 3) return f;   // built (and given its two buffers) on request only
  const size_t word = p->precision == 32 ? 4 : 8;
  f.smem_bytes = 4 * ((size_t)nx + 2 * (size_t)(nx / 64)) * word;
  if (f.smem_bytes + 1024 > 227 * 1024) return f;
  f.threads = nx / 2 < 256 ? nx / 2 : 256;
  int bps = (int)((227 * 1024) / (f.smem_bytes + 1024));
  const int by_regs = p->precision == 32 ? 2048 / 4 / f.threads : 256 / f.threads;   // <= 128 registers (fp32) / 255 (fp64) per thread
  if (bps > by_regs) bps = by_regs;
  if (bps < 1) bps = 1;
  const long long cap = (long long)B200_SMS * bps;
  long long n = cap;
  while (ny / n > 16 && n + cap <= clip::d2q9::FUSED9_MAX_CHUNKS) n += cap;   // more waves rather than chunks of more than 16 rows
  if (n > ny / 2) n = ny / 2 > 0 ? ny / 2 : 1;                                 // at least two rows per chunk
  if (p->tile_chunks >= 1) n = p->tile_chunks < ny ? p->tile_chunks : ny;
  if (n > clip::d2q9::FUSED9_MAX_CHUNKS) n = clip::d2q9::FUSED9_MAX_CHUNKS;
  f.nchunks = (int)n;
  f.part_words = (size_t)f.nchunks * 2 * nx;
  // measured (profiles/r02_experiments.md 4f): correct, 1.036 x the algorithmic DRAM traffic, but issue-bound at two 256-thread blocks per
  // SM: 4096^2 fp32 0.559 ms against 0.524 for k_phi9p + k_step9p, fp64 1.062 against 1.001 -- an option (path = 3), never the default
  f.pays = false;
  f.ok = true;
  return f;
}

Layout make_layout(int nx, int ny, int nz, const clip_params* p) {
  Layout L{};
  L.word = p->precision == 32 ? 4 : 8;
  const size_t n = (size_t)nx * ny * nz, nxy = (size_t)nx * ny;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o += align_up(bytes); return r; };
  const size_t npop = p->lattice == 1 ? 18 : 38;  // f and g of D2Q9 / D3Q19
  L.off_p[0] = take(npop * n * L.word); L.off_p[1] = take(npop * n * L.word);
  L.off_phi = take(n * L.word);
  L.off_u = take(3 * n * L.word);
  const bool outlet = p->bc[5] == CLIP_BC_OUTLET, inlet = p->bc[4] == CLIP_BC_INLET;
  L.off_obf = take(outlet ? 19 * nxy * L.word : 0);
  L.off_obg = take(outlet ? 19 * nxy * L.word : 0);
  L.off_lam = take(outlet ? nxy * L.word : 0);
  L.off_mask = take(inlet ? nxy : 0);
  const FusedPlan fp = fused_plan(nx, ny, nz, p);                // k_fused: second phi buffer + tile-halo partial sums
  const Fused9Plan f9 = fused9_plan(nx, ny, p);                   // the D2Q9 single-pass path: the same two buffers
  L.off_phi2 = take((fp.ok || f9.ok) ? n * L.word : 0);
  L.off_part = take(fp.ok ? fp.part_words * L.word : (f9.ok ? f9.part_words * L.word : 0));
  L.total = o;
  return L;
}

// returns nullptr if valid, else a reason
const char* validate(int nx, int ny, int nz, const clip_params* p) {
  if (!p) return "params is NULL";
  if (nx < 1 || ny < 1 || nz < 1) return "nx, ny, nz must be >= 1";
  if ((double)nx * ny * nz > 2.0e9) return "lattice too large (nx*ny*nz must stay below 2e9)";
  if (p && p->lattice == 1 && ny > 65535) return "D2Q9: ny must stay below 65536 (grid.y of the pair kernels)";
  if (p->precision != 32 && p->precision != 64) return "precision must be 32 or 64";
  if (!(p->rho_h > 0.0) || !(p->rho_l > 0.0)) return "densities must be positive";
  if (!(p->tau_h + 0.5 > 0.0) || !(p->tau_l + 0.5 > 0.0)) return "tau + 1/2 must be positive";
  if (p->visc_interp == 1 && (!(p->tau_h > 0.0) || !(p->tau_l > 0.0))) return "harmonic interpolation needs tau > 0";
  if (p->visc_interp < 0 || p->visc_interp > 2) return "visc_interp must be 0, 1 or 2";
  if (p->collision != CLIP_COLL_WMRT && p->collision != CLIP_COLL_BGK) return "collision must be CLIP_COLL_WMRT (0) or CLIP_COLL_BGK (1)";
  if (p->phase_only != 0 && p->phase_only != 1) return "phase_only must be 0 or 1";
  if (!(3.0 * p->M + 0.5 > 0.0)) return "tau_phi + 1/2 must be positive";
  if (!(p->W > 0.0)) return "W must be positive";
  if (!std::isfinite(p->sigma)) return "sigma must be finite";
  for (int d = 0; d < 3; ++d) {
    const int lo = p->bc[2 * d], hi = p->bc[2 * d + 1];
    if (lo < 0 || lo > 5 || hi < 0 || hi > 5) return "unknown boundary type";
    if (d < 2 && (lo == CLIP_BC_HALO || hi == CLIP_BC_HALO)) return "HALO faces (slab cuts) are only supported on the z faces";
    if ((lo == CLIP_BC_PERIODIC) != (hi == CLIP_BC_PERIODIC)) return "PERIODIC faces must come in pairs";
    const bool open_lo = lo == CLIP_BC_INLET || lo == CLIP_BC_OUTLET, open_hi = hi == CLIP_BC_INLET || hi == CLIP_BC_OUTLET;
    if (d < 2 && (open_lo || open_hi)) return "INLET / OUTLET are only supported on the z faces";
  }
  if (p->bc[4] == CLIP_BC_OUTLET) return "OUTLET is only supported on the +z face";
  if (p->bc[5] == CLIP_BC_INLET) return "INLET is only supported on the -z face";
  if (p->bc[5] == CLIP_BC_OUTLET && nz < 2) return "OUTLET needs nz >= 2";
  if (nz - (p->bc[4] == CLIP_BC_HALO ? 1 : 0) - (p->bc[5] == CLIP_BC_HALO ? 1 : 0) < 2) {
    if (p->bc[4] == CLIP_BC_HALO || p->bc[5] == CLIP_BC_HALO) return "a slab with HALO faces must own at least 2 planes besides its ghost planes";
  }
  if (p->bc[4] == CLIP_BC_INLET && !(p->inlet_r >= 0.0)) return "inlet_r must be >= 0";
  if (p->outlet_u_mode < 0 || p->outlet_u_mode > 2) return "outlet_u_mode must be 0 (U_local), 1 (U_ave) or 2 (U_max)";
  if (p->outlet_clamp != 0 && p->outlet_clamp != 1) return "outlet_clamp must be 0 (B.25 as printed) or 1 (lambda = max(0, U))";
  if (p->outlet_u_time != 0 && p->outlet_u_time != 1) return "outlet_u_time must be 0 (stored u(t)) or 1 (post-stream moment at t+dt)";
  if (p->outlet_u_time == 1 && p->phase_only) return "outlet_u_time = 1 needs the hydrodynamic populations (not phase_only)";
  if (p->path < 0 || p->path > 5) return "path must be 0 (automatic), 1 (generic), 2 (no k_fused), 3 (k_fused where admitted), 4 (k_fused_tma) or 5 (k_fused_tma, g only)";
  if (p->tile_ty != 0 && p->tile_ty != 4 && p->tile_ty != 8 && p->tile_ty != 16) return "tile_ty must be 0 (automatic), 4, 8 or 16";
  if (p->tile_chunks < 0) return "tile_chunks must be >= 0";
  if (p->runtime_nx != 0 && p->runtime_nx != 1) return "runtime_nx must be 0 or 1";
  if (p->cluster_y != 0 && p->cluster_y != 1 && p->cluster_y != 2 && p->cluster_y != 4 && p->cluster_y != 8) return "cluster_y must be 0 (automatic), 1, 2, 4 or 8";
  if (p->lattice != 0 && p->lattice != 1) return "lattice must be 0 (D3Q19) or 1 (D2Q9)";
  if (p->lattice == 1) {
    if (nz != 1 || p->bc[4] != CLIP_BC_PERIODIC || p->bc[5] != CLIP_BC_PERIODIC) return "D2Q9 needs nz = 1 and PERIODIC z faces";
    for (int k = 0; k < 4; ++k)
      if (p->bc[k] != CLIP_BC_PERIODIC && p->bc[k] != CLIP_BC_WALL && p->bc[k] != CLIP_BC_FREESLIP) return "D2Q9 takes PERIODIC, WALL or FREESLIP faces in x and y";
  }
  return nullptr;
}

}  // namespace

struct clip_handle {
  int nx, ny, nz;
  clip_params p;
  Layout L;
  char* ws;
  cudaStream_t stream;
  int cur;      // which of the A/B population buffers holds the current post-collision state
  int phi_cur;  // which phi buffer holds phi(t) (flips only on the k_fused path)
  bool phi_ahead;  // k_fused path: the other phi buffer already holds phi(t+1)
  bool phi_partial[2];  // k_fused path, HALO faces: phi(t+1) of the boundary plane still lacks what the ghost plane sends (clip_halo_unpack)
  int zlo, zhi;    // planes [zlo, zhi) are stepped: all but the ghost planes of HALO faces
  cudaStream_t halo_stream;  // clip_halo_stream: second stream of the overlapped slab step (nullptr: none)
  cudaEvent_t ev_start, ev_bnd, ev_halo;
  bool overlap_open;         // between clip_step_halo_begin and clip_step_halo_end
  bool split_done;           // the last do_step packed the records itself (split launch)
  cudaGraphExec_t gexec;     // GRAPH_STEPS time steps of a small lattice captured as one CUDA graph (step_graphed); nullptr: none
  bool graph_tried;
  long long graph_launches;  // kernel launches inside one replay
  long long graph_steps;     // time steps run by graph replays so far (instrumentation)
  FusedPlan fplan;
  Fused9Plan f9;
  bool inited;
  int mode;            // clip_params.path: 0 = automatic (k_fused + k_fix on wide lattices, else k_phi2 + k_step2), 1 = generic kernels
                       // only, 2 = k_phi2 + k_step2, 3 = k_fused wherever the lattice allows
  int fast_threads;    // threads per block of the pair kernels (128)
  int nx_special;      // nx, or 0 when clip_params.runtime_nx forces the runtime-nx kernels (tests)
  long long launches;
  long long t;
  std::vector<uint8_t> mask_host;
  char err[256];
};

namespace {

template <typename T> clip::KP<T> make_kp(const clip_handle* h) {
  clip::KP<T> P{};
  const clip_params& p = h->p;
  P.nx = h->nx; P.ny = h->ny; P.nz = h->nz;
  P.n = (long long)h->nx * h->ny * h->nz;
  P.nxy = (long long)h->nx * h->ny;
  P.any_nonperiodic = 0;
  for (int k = 0; k < 6; ++k) { P.bc[k] = p.bc[k]; if (p.bc[k] != CLIP_BC_PERIODIC) P.any_nonperiodic = 1; }
  P.z_lo = h->zlo; P.z_cnt = h->zhi - h->zlo; P.z_skip_at = 0; P.z_skip = 0;
  P.has_inlet = p.bc[4] == CLIP_BC_INLET;
  P.has_outlet = p.bc[5] == CLIP_BC_OUTLET;
  P.visc_interp = p.visc_interp;
  P.outlet_u_mode = p.outlet_u_mode; P.outlet_clamp = p.outlet_clamp; P.outlet_u_time = p.outlet_u_time;
  P.collision = p.collision;
  P.phase_only = p.phase_only;
  P.rho_h = (T)p.rho_h; P.rho_l = (T)p.rho_l; P.drho = (T)(p.rho_h - p.rho_l);
  P.tau_h = (T)p.tau_h; P.tau_l = (T)p.tau_l;
  P.rt_h = (T)(p.rho_h * p.tau_h); P.rt_l = (T)(p.rho_l * p.tau_l);
  P.itau_h = (T)(p.tau_h != 0.0 ? 1.0 / p.tau_h : 0.0); P.itau_l = (T)(p.tau_l != 0.0 ? 1.0 / p.tau_l : 0.0);
  P.beta4 = (T)(4.0 * 12.0 * p.sigma / p.W);  // 4 beta, Eq. 12
  P.kappa = (T)(1.5 * p.sigma * p.W);
  P.inv_W = (T)(1.0 / p.W);
  P.om_phi = (T)(1.0 / (3.0 * p.M + 0.5));    // Eq. 33, 37
  P.gx = (T)p.g[0]; P.gy = (T)p.g[1]; P.gz = (T)p.g[2]; P.rho_ref = (T)p.rho_ref;
  for (int k = 0; k < 3; ++k) P.uin[k] = (T)p.inlet_u[k];
  P.phi_in = (T)p.inlet_phi;
  char* ws = h->ws;
  P.p_src = (const T*)(ws + h->L.off_p[h->cur]); P.p_dst = (T*)(ws + h->L.off_p[h->cur ^ 1]);
  P.phi = (T*)(ws + (h->phi_cur ? h->L.off_phi2 : h->L.off_phi)); P.u = (T*)(ws + h->L.off_u);
  P.ob_f = (T*)(ws + h->L.off_obf); P.ob_g = (T*)(ws + h->L.off_obg); P.lam = (T*)(ws + h->L.off_lam);
  P.mask = (const uint8_t*)(ws + h->L.off_mask);
  return P;
}

int check_cuda(clip_handle* h, const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    set_err(h->err, "%s: %s", what, cudaGetErrorString(e));
    return CLIP_ECUDA;
  }
  return CLIP_OK;
}

// 0 = all faces PERIODIC (or open / HALO in z only), 1 = WALL faces, 2 = FREESLIP faces in x / y (instantiations of the pair kernels)
int face_mode(const clip_handle* h) {
  int m = 0;
  for (int k = 0; k < 6; ++k) if (h->p.bc[k] == CLIP_BC_WALL) m = 1;
  for (int k = 0; k < 4; ++k) if (h->p.bc[k] == CLIP_BC_FREESLIP) m = 2;
  return m;
}

unsigned grid_for(long long n, int block) { return (unsigned)((n + block - 1) / block); }

template <typename T> int do_init(clip_handle* h, const void* phi0, const void* u0) {
  h->phi_cur = 0; h->phi_ahead = false; h->phi_partial[0] = h->phi_partial[1] = false;
  h->cur = 1;  // k_init writes into "dst"; flip afterwards so that it becomes the current state
  clip::KP<T> P = make_kp<T>(h);
  if (h->p.lattice == 1) clip::d2q9::k_init9<T><<<grid_for(P.n, 256), 256, 0, h->stream>>>(P, (const T*)phi0, (const T*)u0);
  else clip::k_init<T><<<grid_for(P.n, 256), 256, 0, h->stream>>>(P, (const T*)phi0, (const T*)u0);
  h->launches += 1;
  h->cur = 0;
  return check_cuda(h, "k_init");
}

enum { KIND_PHI = 0, KIND_STEP = 1, KIND_PHI2 = 2, KIND_STEP2 = 3, KIND_FIX = 4, KIND_FUSED = 5, KIND_OUTLET = 6, KIND_COUNT = 7 };
const char* const KIND_NAMES[KIND_COUNT] = {"k_phi", "k_step", "k_phi2", "k_step2", "k_fix", "k_fused", "k_outlet_lam"};

// The pair-per-thread fast kernels (clip_fast.cuh) cover planes whose neighbourhood has only PERIODIC or WALL faces, even nx.
bool fast_ok(const clip_handle* h) {
  if (h->mode == 1 || h->p.lattice != 0) return false;
  if (h->nz > 65535 || h->ny > 65535) return false;  // grid.y / grid.z of the pair kernels
  if (h->p.phase_only) return false;
  if (h->p.collision != CLIP_COLL_WMRT && face_mode(h) == 2) return false;  // BGK with free-slip faces: generic kernels
  if (h->p.bc[4] == CLIP_BC_FREESLIP || h->p.bc[5] == CLIP_BC_FREESLIP) return false;  // free-slip in z: generic kernels only
  // an INLET (-z) / OUTLET (+z) face is served by the generic kernels on its own plane (hybrid launches, do_step)
  return h->nx % 2 == 0 && h->nz >= 4;
}
void fast_shape(const clip_handle* h, dim3& grid, dim3& block) {
  const int pairs = h->nx / 2;
  int bx = 1;
  while (bx < pairs && bx < 128) bx *= 2;
  while (bx > 32 && pairs % bx != 0) bx /= 2;  // e.g. nx = 384: 192 pairs -> 64-wide blocks, no idle threads
  const int by = h->fast_threads / bx > 0 ? h->fast_threads / bx : 1;
  block = dim3(bx, by, 1);
  grid = dim3((pairs + bx - 1) / bx, (h->ny + by - 1) / by, h->nz);
}
template <typename T> clip::FP<T> make_fp(const clip::KP<T>& P) { clip::FP<T> F; F.k = P; return F; }


struct Prof {  // optional per-launch event timing (clip_step_profiled)
  std::vector<cudaEvent_t> ev;
  std::vector<int> kind;
  cudaStream_t stream;
  void begin() { cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, stream); ev.push_back(e); }
  void end(int k) { cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, stream); ev.push_back(e); kind.push_back(k); }
};

bool use_fused(const clip_handle* h) { return fast_ok(h) && h->fplan.ok && (h->mode >= 3 || (h->mode == 0 && h->fplan.pays)); }
bool use_fused9(const clip_handle* h) { return h->p.lattice == 1 && h->f9.ok && (h->mode >= 3 || (h->mode == 0 && h->f9.pays)); }

// lambda of B.25 for the step about to run (k_outlet_lam; the plane-wide schemes of B.22 add a one-block reduction)
template <typename T> void outlet_lambda(clip_handle* h, const clip::KP<T>& P, Prof* prof) {
  if (prof) prof->begin();
  clip::k_outlet_lam<T><<<grid_for(P.nxy, 256), 256, 0, h->stream>>>(P);
  h->launches += 1;
  if (P.outlet_u_mode != 0) { clip::k_outlet_reduce<T><<<1, 1024, 0, h->stream>>>(P); h->launches += 1; }
  if (prof) prof->end(KIND_OUTLET);
}

// k_fused path on a lattice with an INLET / OUTLET z face, from the state (f+, g+, u) at the current time t: lambda of B.25 for the
// step t -> t+1 and phi(t+1) of the planes the single-pass kernel cannot complete -- the open planes themselves (inlet rule,
// B.26-B.27) and their neighbours, which receive g+ from them -- by the generic k_phi, into the phi(t+1) buffer.
template <typename T> void fused_open_planes(clip_handle* h, Prof* prof) {
  const int glo = h->p.bc[4] == CLIP_BC_INLET ? 1 : 0, ghi = h->p.bc[5] == CLIP_BC_OUTLET ? 1 : 0;
  if (!glo && !ghi) return;
  clip::KP<T> P = make_kp<T>(h);
  P.phi = (T*)(h->ws + (h->phi_cur ? h->L.off_phi : h->L.off_phi2));
  if (P.has_outlet) outlet_lambda<T>(h, P, prof);
  clip::KP<T> Q = P;   // planes 0, 1 and / or nz-2, nz-1 in one launch
  Q.z_lo = glo ? 0 : h->nz - 2; Q.z_cnt = 2 * (glo + ghi);
  if (glo && ghi) { Q.z_skip_at = 2; Q.z_skip = h->nz - 4; }
  if (prof) prof->begin();
  clip::k_phi<T><<<grid_for(Q.z_cnt * P.nxy, 256), 256, 0, h->stream>>>(Q);
  if (prof) prof->end(KIND_PHI);
  h->launches += 1;
}

// k_fused path, once after clip_init: phi(t+1) = sum_a g+_a(x - e_a, t) into the second phi buffer (one k_phi2 launch, plus the
// generic kernel on the planes next to an open face).
template <typename T> void fused_prepass(clip_handle* h, Prof* prof) {
  if (h->phi_ahead) return;
  const int faces = face_mode(h);
  const int glo = h->p.bc[4] == CLIP_BC_INLET ? 1 : 0, ghi = h->p.bc[5] == CLIP_BC_OUTLET ? 1 : 0;
  dim3 fg, fb;
  fast_shape(h, fg, fb);
  clip::FP<T> F = make_fp<T>(make_kp<T>(h));
  F.k.phi = (T*)(h->ws + (h->phi_cur ? h->L.off_phi : h->L.off_phi2));
  F.k.z_lo = h->zlo + glo; F.k.z_cnt = h->zhi - ghi - F.k.z_lo; fg.z = (unsigned)F.k.z_cnt;
  if (prof) prof->begin();
  clip::launch_phi2<T>(faces, h->nx_special, fg, fb, h->stream, F);
  if (prof) prof->end(KIND_PHI2);
  h->launches += 1;
  fused_open_planes<T>(h, prof);
  h->phi_ahead = true;
}

// split = true (clip_step_halo_begin, one step, k_fused path with >= 3 chunks): the first and the last z chunk -- the ones next to
// the HALO faces -- run on the halo stream, followed there by the pack kernel (the caller's exchange then overlaps the interior
// chunks, which run on the handle's stream together with k_fix).
template <typename T> int do_step(clip_handle* h, int nsteps, Prof* prof = nullptr, bool split = false, void* d_lo = nullptr, void* d_hi = nullptr) {
  const bool fast = fast_ok(h);
  const int faces = face_mode(h);
  const bool xwalls = h->p.bc[0] != CLIP_BC_PERIODIC;
  dim3 fg, fb;
  if (fast) fast_shape(h, fg, fb);
  const bool fused = use_fused(h);
  const bool plain = h->p.collision == CLIP_COLL_WMRT && !h->p.phase_only;   // k_step<T, true>: no mode tests in the direction loop
  for (int s = 0; s < nsteps; ++s) {
    clip::KP<T> P = make_kp<T>(h);
    if (use_fused9(h)) {  // D2Q9, one pass over f and g (clip_d2q9.cuh): the state is that of the k_fused path below
      const Fused9Plan& f9 = h->f9;
      T* const phi_now = (T*)(h->ws + (h->phi_cur ? h->L.off_phi2 : h->L.off_phi));
      T* const phi_next = (T*)(h->ws + (h->phi_cur ? h->L.off_phi : h->L.off_phi2));
      const dim3 g9((h->nx / 2 + 127) / 128, h->ny);
      if (!h->phi_ahead) {   // once after clip_init: phi(t+1) = sum_a g+_a(x - e_a, t)
        clip::KP<T> Q = P;
        Q.phi = phi_next;
        if (prof) prof->begin();
        clip::d2q9::k_phi9p<T><<<g9, 128, 0, h->stream>>>(Q);
        if (prof) prof->end(KIND_PHI2);
        h->launches += 1;
        h->phi_ahead = true;
      }
      clip::KP<T> Q = P;
      Q.phi = phi_next;
      clip::d2q9::Fused9P<T> U9;
      U9.phi_dst = phi_now; U9.part = (T*)(h->ws + h->L.off_part); U9.nchunks = f9.nchunks;
      auto kern = clip::d2q9::k_fused9<T>;
      constexpr int DEV_MAX = 64;
      static bool attr9[DEV_MAX] = {};   // the shared-memory opt-in is per device (and per T: do_step<T>)
      int dev = 0;
      cudaGetDevice(&dev);
      if (dev < 0 || dev >= DEV_MAX || !attr9[dev]) {
        const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
        if (e != cudaSuccess) { set_err(h->err, "k_fused9: %s", cudaGetErrorString(e)); return CLIP_ECUDA; }
        if (dev >= 0 && dev < DEV_MAX) attr9[dev] = true;
      }
      if (prof) prof->begin();
      kern<<<f9.nchunks, f9.threads, f9.smem_bytes, h->stream>>>(Q, U9);
      if (prof) { prof->end(KIND_FUSED); prof->begin(); }
      clip::d2q9::k_fix9<T><<<dim3(f9.nchunks, (h->nx / 2 + 127) / 128), 128, 0, h->stream>>>(Q, U9);
      if (prof) prof->end(KIND_FIX);
      h->launches += 2;
      h->cur ^= 1;
      h->phi_cur ^= 1;
      h->t += 1;
      continue;
    }
    if (fused) {  // one pass over f and g (clip_fused.cuh) + the tile-surface fix-up of phi(t+2)
      // State between fused steps: populations f+(t), g+(t); phi buffer `phi_cur` = phi(t) (what clip_get returns), the
      // other buffer = phi(t+1) = sum_a g+_a(x - e_a, t), which the collision at t+1 needs (first step: one k_phi2).
      const FusedPlan& fp = h->fplan;
      clip::FP<T> F = make_fp<T>(P);
      T* const phi_now = (T*)(h->ws + (h->phi_cur ? h->L.off_phi2 : h->L.off_phi));
      T* const phi_next = (T*)(h->ws + (h->phi_cur ? h->L.off_phi : h->L.off_phi2));
      F.k.phi = phi_next;
      fused_prepass<T>(h, prof);
      {  // the INLET / OUTLET planes (one launch for both): generic kernel, phi(t+1) and lambda are in place
        const int olo = h->p.bc[4] == CLIP_BC_INLET ? 1 : 0, ohi = h->p.bc[5] == CLIP_BC_OUTLET ? 1 : 0;
        if (olo + ohi) {
          clip::KP<T> Q = F.k;
          Q.z_lo = olo ? 0 : h->nz - 1; Q.z_cnt = olo + ohi;
          if (olo && ohi) { Q.z_skip_at = 1; Q.z_skip = h->nz - 2; }
          if (prof) prof->begin();
          clip::k_step<T, true><<<grid_for(Q.z_cnt * P.nxy, 256), 256, 0, h->stream>>>(Q);   // the k_fused path is WMRT, two-phase
          if (prof) prof->end(KIND_STEP);
          h->launches += 1;
        }
      }
      clip::FusedP<T> U;
      U.z_wrap = h->p.bc[4] == CLIP_BC_PERIODIC ? 1 : 0;
      U.phi_dst = phi_now;  // becomes phi(t+2); phi(t) is no longer needed once the time is t+1
      U.part = (T*)(h->ws + h->L.off_part);
      U.ty = fp.ty; U.ytiles = fp.ytiles; U.nchunks = fp.nchunks; U.tzmax = fp.tzmax;
      for (int c = 0; c <= fp.nchunks; ++c) U.zc[c] = fp.zc[c];
      U.tile_stride = (long long)(2 * fp.tzmax + 2 * (fp.ty + 2)) * h->nx;
      U.cs = 1;
      if (prof) prof->begin();
      cudaError_t fe;
      if (split && !fp.tma && fp.nchunks >= 3 && fp.zc[1] - fp.zc[0] >= 2 && fp.zc[fp.nchunks] - fp.zc[fp.nchunks - 1] >= 2) {
        h->split_done = true;
        cudaEventRecord(h->ev_start, h->stream);
        cudaStreamWaitEvent(h->halo_stream, h->ev_start, 0);
        U.c_mode = 1;
        fe = clip::launch_fused<T>(faces, h->nx_special, dim3(fp.ytiles, 2), dim3(fp.threads), fp.smem_bytes, h->halo_stream, F, U);
        cudaEventRecord(h->ev_bnd, h->halo_stream);
        if (fe == cudaSuccess) {  // the records need the new populations of the boundary planes and their neighbours only
          const cudaStream_t main_stream = h->stream;
          h->cur ^= 1; h->stream = h->halo_stream;
          const int rc = clip_halo_pack(h, d_lo, d_hi);
          h->cur ^= 1; h->stream = main_stream;
          if (rc != CLIP_OK) return rc;
          U.c_mode = 2;
          fe = clip::launch_fused<T>(faces, h->nx_special, dim3(fp.ytiles, fp.nchunks - 2), dim3(fp.threads), fp.smem_bytes, h->stream, F, U);
          h->launches += 1;
        }
        cudaStreamWaitEvent(h->stream, h->ev_bnd, 0);
      } else if (fp.cs > 1) {   // thread-block clusters of fp.cs y-adjacent tiles; k_fix (same U) skips the surfaces they share
        U.c_mode = 0; U.cs = fp.cs;
        fe = clip::launch_fused_cl<T>(faces, h->nx_special, dim3(fp.ytiles, fp.nchunks), dim3(fp.threads), fp.smem_bytes, h->stream, F, U);
        if (fe != cudaSuccess) {  // a device / partition that cannot place the cluster: the plain kernel from now on (same results)
          cudaGetLastError();
          h->fplan.cs = 1; U.cs = 1;
          fe = clip::launch_fused<T>(faces, h->nx_special, dim3(fp.ytiles, fp.nchunks), dim3(fp.threads), fp.smem_bytes, h->stream, F, U);
        }
      } else {
        U.c_mode = 0;
        if (fp.tma) fe = clip::launch_fused_tma<T>(h->nx_special, fp.tma_g, dim3(fp.ytiles, fp.nchunks), dim3(fp.threads), fp.smem_bytes, h->stream, F, U);
        else fe = clip::launch_fused<T>(faces, h->nx_special, dim3(fp.ytiles, fp.nchunks), dim3(fp.threads), fp.smem_bytes, h->stream, F, U);
      }
      if (fe != cudaSuccess) { set_err(h->err, "k_fused: %s", cudaGetErrorString(fe)); return CLIP_ECUDA; }
      if (prof) { prof->end(KIND_FUSED); prof->begin(); }
      const int fix_rpb = clip::FIX_ROWS * (clip::FIX_THREADS / clip::fix_threads_per_row(h->nx, clip::Vec16<T>::EV));  // rows per block
      clip::launch_fix<T>(dim3(fp.ytiles, fp.nchunks, (2 * fp.tzmax + 2 * (fp.ty - 2) + fix_rpb - 1) / fix_rpb), h->stream, F, U);
      if (prof) prof->end(KIND_FIX);
      h->launches += 2;
      h->cur ^= 1;
      h->phi_cur ^= 1;
      h->t += 1;
      h->phi_partial[0] = h->p.bc[4] == CLIP_BC_HALO; h->phi_partial[1] = h->p.bc[5] == CLIP_BC_HALO;  // completed by clip_halo_unpack
      fused_open_planes<T>(h, prof);  // open z faces: lambda and the boundary planes of phi(t+2), from the new state
      continue;
    }
    // planes next to an INLET / OUTLET face: generic kernels; all other planes: pair kernels (when the lattice allows)
    const int glo = (fast && h->p.bc[4] == CLIP_BC_INLET) ? 1 : 0, ghi = (fast && h->p.bc[5] == CLIP_BC_OUTLET) ? 1 : 0;
    clip::KP<T> Pface = P;   // the planes z = 0 and / or nz-1, one launch
    Pface.z_lo = glo ? 0 : h->nz - 1; Pface.z_cnt = glo + ghi;
    if (glo && ghi) { Pface.z_skip_at = 1; Pface.z_skip = h->nz - 2; }
    clip::FP<T> F;
    if (fast) { F = make_fp<T>(P); F.k.z_lo = h->zlo + glo; F.k.z_cnt = h->zhi - ghi - F.k.z_lo; fg.z = (unsigned)F.k.z_cnt; }
    if (P.has_outlet) outlet_lambda<T>(h, P, prof);  // lambda of B.25 for this step, before anything of the step reads it
    for (int pass = 0; pass < 2; ++pass) {  // pass 0: phi(t+1); pass 1: macros + collisions
      if (!fast) {
        if (prof) prof->begin();
        if (h->p.lattice == 1 && h->nx % 2 == 0 && h->mode != 1) {  // D2Q9, pair-per-thread packed kernels (clip_d2q9.cuh)
          int bx = 1;
          while (bx < h->nx / 2 && bx < 128) bx *= 2;
          const dim3 g9((h->nx / 2 + bx - 1) / bx, h->ny);
          if (pass == 0) clip::d2q9::k_phi9p<T><<<g9, bx, 0, h->stream>>>(P);
          else clip::d2q9::k_step9p<T><<<g9, bx, 0, h->stream>>>(P);
        } else if (h->p.lattice == 1) {  // D2Q9, thread per node (odd nx, path 1)
          if (pass == 0) clip::d2q9::k_phi9<T><<<grid_for(P.n, 256), 256, 0, h->stream>>>(P);
          else clip::d2q9::k_step9<T><<<grid_for(P.n, 256), 256, 0, h->stream>>>(P);
        } else if (pass == 0) clip::k_phi<T><<<grid_for(P.z_cnt * P.nxy, 256), 256, 0, h->stream>>>(P);
        else if (plain) clip::k_step<T, true><<<grid_for(P.z_cnt * P.nxy, 256), 256, 0, h->stream>>>(P);
        else clip::k_step<T><<<grid_for(P.z_cnt * P.nxy, 256), 256, 0, h->stream>>>(P);
        h->launches += 1;
        if (prof) prof->end(pass == 0 ? KIND_PHI : KIND_STEP);
        continue;
      }
      if (glo + ghi) {
        const clip::KP<T>& Q = Pface;
        if (prof) prof->begin();
        if (pass == 0) clip::k_phi<T><<<grid_for(Q.z_cnt * P.nxy, 256), 256, 0, h->stream>>>(Q);
        else if (plain) clip::k_step<T, true><<<grid_for(Q.z_cnt * P.nxy, 256), 256, 0, h->stream>>>(Q);
        else clip::k_step<T><<<grid_for(Q.z_cnt * P.nxy, 256), 256, 0, h->stream>>>(Q);
        h->launches += 1;
        if (prof) prof->end(pass == 0 ? KIND_PHI : KIND_STEP);
      }
      if (prof) prof->begin();
      if (pass == 0) {
        clip::launch_phi2<T>(faces, h->nx_special, fg, fb, h->stream, F);
      } else {
        clip::launch_step2<T>(faces, xwalls, h->nx_special, fg, fb, h->stream, F);
      }
      h->launches += 1;
      if (prof) prof->end(pass == 0 ? KIND_PHI2 : KIND_STEP2);
    }
    h->cur ^= 1;
    h->t += 1;
  }
  return check_cuda(h, "k_step");
}

template <typename T> int do_get(clip_handle* h, void* phi, void* p, void* u) {
  clip::KP<T> P = make_kp<T>(h);
  if (h->p.lattice == 1) clip::d2q9::k_get9<T><<<grid_for(P.n, 256), 256, 0, h->stream>>>(P, (T*)phi, (T*)p, (T*)u);
  else clip::k_get<T><<<grid_for(P.n, 256), 256, 0, h->stream>>>(P, (T*)phi, (T*)p, (T*)u);
  h->launches += 1;
  return check_cuda(h, "k_get");
}

// z-slab decomposition (clip.h).  A HALO z face means: the first / last plane of this lattice is a GHOST plane, an
// image of the neighbouring slab's outermost owned plane; the step kernels cover the owned planes only.  What an owned plane
// reads from the ghost plane next to it: the 5 + 5 populations that move towards it (pull streaming, Alg. 2) and phi of the
// next collision (stencils of Eq. 40).  The record one slab sends per face node (12 words, SURVEY's 10 + 1 and one more):
//   [0..4]  f+_a, [5..9] g+_a of its boundary plane B for the five a that point at the neighbour (e_z = s)
//   [10]    the PART of phi_B(next) = sum_a g_a (Eq. 38 after streaming) that comes from its own side (planes B, B -+ 1; links
//           bounced at an x / y wall included)
//   [11]    C = what B sends INTO the neighbour's boundary plane: sum over the five a of g+_a(x - e_a), in-plane faces applied
// The receiver completes both boundary planes by additions: phi_ghost = record[10] + (its own C, which it has just sent), and --
// on the k_fused path, whose scatter could not see the ghost's populations -- phi_B += record[11].
template <typename T, int a = 1> struct HaloDirs {
  // sums over directions of the pull at node (pb, nb); WHICH selects by e_z: +1 / -1 = only that sign; 0 handled by the caller
  static __device__ __forceinline__ void run(const clip::KP<T>& P, long long pb, const clip::Nbr& nb, int s, T& part, T& c_in) {
    using namespace clip;
    const bool bounced = src_bounce<a>(nb);
    // partial of the boundary plane: everything except what comes from beyond the HALO face (e_z = -s, not bounced in-plane)
    if (cz(a) != 0) {
      if (cz(a) != -s || bounced) part += pull_one<T, a>(P.p_src + Q * P.nx, P.nx, pb, nb, nb.any);
    } else part += pull_one<T, a>(P.p_src + Q * P.nx, P.nx, pb, nb, nb.any);
    HaloDirs<T, a + 1>::run(P, pb, nb, s, part, c_in);
  }
  static __device__ __forceinline__ void into(const clip::KP<T>& P, long long pbg, const clip::Nbr& ng, int s, T& c) {
    using namespace clip;
    if (cz(a) != 0 && cz(a) == s && !src_bounce<a>(ng)) c += pull_one<T, a>(P.p_src + Q * P.nx, P.nx, pbg, ng, ng.any);
    HaloDirs<T, a + 1>::into(P, pbg, ng, s, c);
  }
  static __device__ __forceinline__ void copy_out(const clip::KP<T>& P, long long pb, int s, T* rec, long long c, int& k) {
    using namespace clip;
    if (cz(a) == s) { rec[k * P.nxy + c] = P.p_src[pb + a * P.nx]; rec[(5 + k) * P.nxy + c] = P.p_src[pb + (Q + a) * P.nx]; ++k; }
    HaloDirs<T, a + 1>::copy_out(P, pb, s, rec, c, k);
  }
  static __device__ __forceinline__ void copy_in(const clip::KP<T>& P, T* pop, long long pb, int s, const T* rec, long long c, int& k) {
    using namespace clip;
    if (cz(a) == s) { pop[pb + a * P.nx] = rec[k * P.nxy + c]; pop[pb + (Q + a) * P.nx] = rec[(5 + k) * P.nxy + c]; ++k; }
    HaloDirs<T, a + 1>::copy_in(P, pop, pb, s, rec, c, k);
  }
};
template <typename T> struct HaloDirs<T, clip::Q> {
  static __device__ __forceinline__ void run(const clip::KP<T>&, long long, const clip::Nbr&, int, T&, T&) {}
  static __device__ __forceinline__ void into(const clip::KP<T>&, long long, const clip::Nbr&, int, T&) {}
  static __device__ __forceinline__ void copy_out(const clip::KP<T>&, long long, int, T*, long long, int&) {}
  static __device__ __forceinline__ void copy_in(const clip::KP<T>&, T*, long long, int, const T*, long long, int&) {}
};
constexpr int HALO_WORDS = 12;

// grid = (ceil(nxy / 256), 2): blockIdx.y = side (0: -z, 1: +z); a side without a record has rec == nullptr
template <typename T> __global__ void __launch_bounds__(256) k_halo_pack(const __grid_constant__ clip::KP<T> P, T* rec_lo, T* rec_hi) {
  using namespace clip;
  const int side = blockIdx.y;
  T* const rec = side ? rec_hi : rec_lo;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (!rec || c >= P.nxy) return;
  const int x = (int)(c % P.nx), y = (int)(c / P.nx);
  const int s = side ? 1 : -1, zg = side ? P.nz - 1 : 0, zb = zg - s;
  const long long ib = (long long)zb * P.nxy + c, ig = (long long)zg * P.nxy + c;
  const long long pb = pop_base(ib, x), pbg = pop_base(ig, x);
  int k = 0;
  HaloDirs<T>::copy_out(P, pb, s, rec, c, k);
  // the boundary plane is never the first / last plane of the array, so its Nbr (in-plane faces, plain z offsets) also serves
  // the pull of the ghost-plane node from this side
  const Nbr nb = make_nbr(P, x, y, zb);
  const Nbr& ng = nb;
  T part = P.p_src[pb + Q * P.nx], dummy = T(0), cin = T(0);  // direction 0
  HaloDirs<T>::run(P, pb, nb, s, part, dummy);
  HaloDirs<T>::into(P, pbg, ng, s, cin);
  if (P.has_inlet && zb == 0 && P.mask[c]) part = P.phi_in;   // (cannot happen: an inlet plane is never next to a HALO face)
  rec[10 * P.nxy + c] = part;
  rec[11 * P.nxy + c] = cin;
}
// recv_*: the record the neighbour on that side packed (its opposite side); sent_*: the record this handle packed for that side
template <typename T> __global__ void __launch_bounds__(256)
k_halo_unpack(const __grid_constant__ clip::KP<T> P, const T* recv_lo, const T* recv_hi, const T* sent_lo, const T* sent_hi, T* phi_next,
              int add_lo, int add_hi) {
  using namespace clip;
  const int side = blockIdx.y;
  const T* const recv = side ? recv_hi : recv_lo;
  const T* const sent = side ? sent_hi : sent_lo;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (!recv || c >= P.nxy) return;
  const int x = (int)(c % P.nx);
  const int s = side ? 1 : -1, zg = side ? P.nz - 1 : 0, zb = zg - s;
  const long long ib = (long long)zb * P.nxy + c, ig = (long long)zg * P.nxy + c;
  int k = 0;
  HaloDirs<T>::copy_in(P, const_cast<T*>(P.p_src), pop_base(ig, x), -s, recv, c, k);   // what moves from the neighbour towards me
  phi_next[ig] = recv[10 * P.nxy + c] + sent[11 * P.nxy + c];
  if (side ? add_hi : add_lo) phi_next[ib] += recv[11 * P.nxy + c];
}

// Small lattices are launch-bound (64^3: two launches of ~5 and ~10 us per step): clip_step(n) replays GRAPH_STEPS steps as ONE CUDA
// graph (SURVEY.md:121).  The A/B buffers return to the same roles after an even number of steps, so one graph captured at parity 0
// serves every replay; kernel parameters (device pointers into the caller's workspace, sizes) are frozen in it.  Only on a stream that
// can be captured (not the legacy default stream, not a stream the caller is capturing), without HALO faces, up to 4 M nodes.
constexpr int GRAPH_STEPS = 16;
bool graph_eligible(const clip_handle* h) {
  if ((long long)h->nx * h->ny * h->nz > (1LL << 22)) return false;
  if (h->p.bc[4] == CLIP_BC_HALO || h->p.bc[5] == CLIP_BC_HALO) return false;
  if (h->stream == nullptr || h->stream == cudaStreamLegacy || h->stream == cudaStreamPerThread) return false;
  cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(h->stream, &st) != cudaSuccess) { cudaGetLastError(); return false; }
  return st == cudaStreamCaptureStatusNone;
}
template <typename T> int step_graphed(clip_handle* h, int n) {
  if (n < 2 * GRAPH_STEPS || (h->graph_tried && !h->gexec) || !graph_eligible(h)) return do_step<T>(h, n);
  // reach the state the graph is (to be) captured in: buffer parity 0 and, on the k_fused path, phi(t+1) in place
  while (n > 0 && (h->cur != 0 || ((use_fused(h) || use_fused9(h)) && !h->phi_ahead))) {
    const int rc = do_step<T>(h, 1);
    if (rc != CLIP_OK) return rc;
    --n;
  }
  if (!h->gexec && n >= GRAPH_STEPS) {
    h->graph_tried = true;
    const long long t0 = h->t, l0 = h->launches;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      const int rc = do_step<T>(h, GRAPH_STEPS);     // recorded, not run: the host-side counters are put back below
      const cudaError_t e = cudaStreamEndCapture(h->stream, &graph);
      h->graph_launches = h->launches - l0;
      h->t = t0; h->launches = l0;                   // cur / phi_cur are back at parity 0 after an even number of steps
      if (rc == CLIP_OK && e == cudaSuccess && graph && cudaGraphInstantiate(&h->gexec, graph, 0) != cudaSuccess) h->gexec = nullptr;
      if (graph) cudaGraphDestroy(graph);
    }
    cudaGetLastError();  // a failed capture is not an error of the step: plain launches follow
  }
  while (h->gexec && n >= GRAPH_STEPS) {
    if (cudaGraphLaunch(h->gexec, h->stream) != cudaSuccess) { set_err(h->err, "clip_step: graph launch: %s", cudaGetErrorString(cudaGetLastError())); return CLIP_ECUDA; }
    h->t += GRAPH_STEPS; h->launches += h->graph_launches; h->graph_steps += GRAPH_STEPS;
    n -= GRAPH_STEPS;
  }
  return do_step<T>(h, n);
}

}  // namespace

extern "C" {

size_t clip_halo_bytes(const clip_t* h) {
  if (!h) return 0;
  return (size_t)h->nx * h->ny * h->L.word * HALO_WORDS;
}
int clip_halo_pack(clip_t* h, void* d_lo, void* d_hi) {
  if (!h) return CLIP_EINVAL;
  if (!h->inited) { set_err(h->err, "clip_halo_pack: clip_init has not been called"); return CLIP_ESTATE; }
  const bool lo = h->p.bc[4] == CLIP_BC_HALO, hi = h->p.bc[5] == CLIP_BC_HALO;
  if ((lo && !d_lo) || (hi && !d_hi) || ((uintptr_t)d_lo) % 16 || ((uintptr_t)d_hi) % 16) {
    set_err(h->err, "clip_halo_pack: every HALO face needs a 16-byte aligned device buffer of clip_halo_bytes");
    return CLIP_EINVAL;
  }
  if (!lo && !hi) return CLIP_OK;
  const dim3 grid(grid_for((long long)h->nx * h->ny, 256), 2);
  if (h->p.precision == 32) k_halo_pack<float><<<grid, 256, 0, h->stream>>>(make_kp<float>(h), lo ? (float*)d_lo : nullptr, hi ? (float*)d_hi : nullptr);
  else k_halo_pack<double><<<grid, 256, 0, h->stream>>>(make_kp<double>(h), lo ? (double*)d_lo : nullptr, hi ? (double*)d_hi : nullptr);
  h->launches += 1;
  return check_cuda(h, "clip_halo_pack");
}
int clip_halo_unpack(clip_t* h, const void* d_recv_lo, const void* d_recv_hi, const void* d_sent_lo, const void* d_sent_hi) {
  if (!h) return CLIP_EINVAL;
  if (!h->inited) { set_err(h->err, "clip_halo_unpack: clip_init has not been called"); return CLIP_ESTATE; }
  const bool lo = h->p.bc[4] == CLIP_BC_HALO, hi = h->p.bc[5] == CLIP_BC_HALO;
  if ((lo && (!d_recv_lo || !d_sent_lo)) || (hi && (!d_recv_hi || !d_sent_hi)) || ((uintptr_t)d_recv_lo) % 16 || ((uintptr_t)d_recv_hi) % 16 ||
      ((uintptr_t)d_sent_lo) % 16 || ((uintptr_t)d_sent_hi) % 16) {
    set_err(h->err, "clip_halo_unpack: every HALO face needs the received and the sent record (16-byte aligned device buffers)");
    return CLIP_EINVAL;
  }
  if (!lo && !hi) return CLIP_OK;
  const dim3 grid(grid_for((long long)h->nx * h->ny, 256), 2);
  // phi of the NEXT collision: the k_fused path keeps it in the second buffer, the other paths rewrite the one buffer in place
  char* const next = h->ws + (use_fused(h) ? (h->phi_cur ? h->L.off_phi : h->L.off_phi2) : h->L.off_phi);
  const int add_lo = lo && h->phi_partial[0], add_hi = hi && h->phi_partial[1];
  if (h->p.precision == 32)
    k_halo_unpack<float><<<grid, 256, 0, h->stream>>>(make_kp<float>(h), lo ? (const float*)d_recv_lo : nullptr, hi ? (const float*)d_recv_hi : nullptr,
                                                      (const float*)d_sent_lo, (const float*)d_sent_hi, (float*)next, add_lo, add_hi);
  else
    k_halo_unpack<double><<<grid, 256, 0, h->stream>>>(make_kp<double>(h), lo ? (const double*)d_recv_lo : nullptr, hi ? (const double*)d_recv_hi : nullptr,
                                                       (const double*)d_sent_lo, (const double*)d_sent_hi, (double*)next, add_lo, add_hi);
  h->phi_partial[0] = h->phi_partial[1] = false;
  h->launches += 1;
  return check_cuda(h, "clip_halo_unpack");
}

int clip_halo_stream(clip_t* h, void* cuda_stream) {
  if (!h) return CLIP_EINVAL;
  if (h->overlap_open) { set_err(h->err, "clip_halo_stream: a step is open (clip_step_halo_end missing)"); return CLIP_ESTATE; }
  if (cuda_stream && !h->ev_start) {
    if (cudaEventCreateWithFlags(&h->ev_start, cudaEventDisableTiming) != cudaSuccess || cudaEventCreateWithFlags(&h->ev_bnd, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_halo, cudaEventDisableTiming) != cudaSuccess) {
      set_err(h->err, "clip_halo_stream: %s", cudaGetErrorString(cudaGetLastError()));
      return CLIP_ECUDA;
    }
  }
  h->halo_stream = (cudaStream_t)cuda_stream;
  return CLIP_OK;
}
int clip_step_halo_begin(clip_t* h, void* d_lo, void* d_hi) {
  if (!h) return CLIP_EINVAL;
  if (!h->inited) { set_err(h->err, "clip_step_halo_begin: clip_init has not been called"); return CLIP_ESTATE; }
  if (!h->halo_stream) { set_err(h->err, "clip_step_halo_begin: no halo stream (clip_halo_stream)"); return CLIP_ESTATE; }
  if (h->overlap_open) { set_err(h->err, "clip_step_halo_begin: the previous step is still open (clip_step_halo_end missing)"); return CLIP_ESTATE; }
  const bool lo = h->p.bc[4] == CLIP_BC_HALO, hi = h->p.bc[5] == CLIP_BC_HALO;
  if ((lo && !d_lo) || (hi && !d_hi) || ((uintptr_t)d_lo) % 16 || ((uintptr_t)d_hi) % 16) {
    set_err(h->err, "clip_step_halo_begin: every HALO face needs a 16-byte aligned device buffer of clip_halo_bytes");
    return CLIP_EINVAL;
  }
  h->split_done = false;
  int rc = h->p.precision == 32 ? do_step<float>(h, 1, nullptr, use_fused(h), d_lo, d_hi) : do_step<double>(h, 1, nullptr, use_fused(h), d_lo, d_hi);
  if (rc != CLIP_OK) return rc;
  if (!h->split_done) {  // other paths: the whole step on the handle's stream, then the records on the halo stream
    cudaEventRecord(h->ev_start, h->stream);
    cudaStreamWaitEvent(h->halo_stream, h->ev_start, 0);
    const cudaStream_t main_stream = h->stream;
    h->stream = h->halo_stream;
    rc = clip_halo_pack(h, d_lo, d_hi);
    h->stream = main_stream;
    if (rc != CLIP_OK) return rc;
  }
  h->overlap_open = true;
  return check_cuda(h, "clip_step_halo_begin");
}
int clip_step_halo_end(clip_t* h, const void* d_recv_lo, const void* d_recv_hi, const void* d_sent_lo, const void* d_sent_hi) {
  if (!h) return CLIP_EINVAL;
  if (!h->overlap_open) { set_err(h->err, "clip_step_halo_end: no open step (clip_step_halo_begin)"); return CLIP_ESTATE; }
  cudaEventRecord(h->ev_halo, h->halo_stream);     // after the caller's exchange
  cudaStreamWaitEvent(h->stream, h->ev_halo, 0);
  h->overlap_open = false;
  return clip_halo_unpack(h, d_recv_lo, d_recv_hi, d_sent_lo, d_sent_hi);
}

size_t clip_workspace_bytes(int nx, int ny, int nz, const clip_params* params) {
  const char* why = validate(nx, ny, nz, params);
  if (why) { set_err(g_create_error, "clip_workspace_bytes: %s", why); return 0; }
  return make_layout(nx, ny, nz, params).total;
}

int clip_create(clip_t** out, int nx, int ny, int nz, const clip_params* params, void* d_workspace, size_t bytes,
                void* cuda_stream) {
  if (!out) { set_err(g_create_error, "clip_create: out is NULL"); return CLIP_EINVAL; }
  *out = nullptr;
  const char* why = validate(nx, ny, nz, params);
  if (why) { set_err(g_create_error, "clip_create: %s", why); return CLIP_EINVAL; }
  if (!d_workspace) { set_err(g_create_error, "clip_create: workspace is NULL"); return CLIP_EINVAL; }
  if (((uintptr_t)d_workspace) % ALIGN) { set_err(g_create_error, "clip_create: workspace must be 256-byte aligned"); return CLIP_EINVAL; }
  Layout L = make_layout(nx, ny, nz, params);
  if (bytes < L.total) {
    set_err(g_create_error, "clip_create: workspace too small (%zu < %zu bytes)", bytes, L.total);
    return CLIP_ENOMEM;
  }
  clip_handle* h = new (std::nothrow) clip_handle();
  if (!h) { set_err(g_create_error, "clip_create: out of host memory"); return CLIP_ENOMEM; }
  h->nx = nx; h->ny = ny; h->nz = nz; h->p = *params; h->L = L; h->ws = (char*)d_workspace;
  h->stream = (cudaStream_t)cuda_stream; h->cur = 0; h->phi_cur = 0; h->phi_ahead = false; h->inited = false;
  h->phi_partial[0] = h->phi_partial[1] = false;
  h->halo_stream = nullptr; h->ev_start = h->ev_bnd = h->ev_halo = nullptr; h->overlap_open = false; h->split_done = false;
  h->gexec = nullptr; h->graph_tried = false; h->graph_launches = 0; h->graph_steps = 0;
  h->zlo = params->bc[4] == CLIP_BC_HALO ? 1 : 0; h->zhi = nz - (params->bc[5] == CLIP_BC_HALO ? 1 : 0);
  h->fplan = fused_plan(nx, ny, nz, params);
  h->f9 = fused9_plan(nx, ny, params);
  h->mode = params->path;
  h->fast_threads = 128;  // measured: fp64 8.2 vs 7.6 GLUPS, fp32 (with 3 blocks per SM) +2 % against 256-thread blocks
  h->nx_special = params->runtime_nx ? 0 : nx;
  h->launches = 0; h->t = 0; h->err[0] = 0;
  if (params->bc[4] == CLIP_BC_INLET) {  // disc mask, decided in double on the host
    h->mask_host.resize((size_t)nx * ny);
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        const double dx = x - params->inlet_c[0], dy = y - params->inlet_c[1];
        h->mask_host[(size_t)y * nx + x] = (dx * dx + dy * dy <= params->inlet_r * params->inlet_r) ? 1 : 0;
      }
    cudaError_t e = cudaMemcpyAsync(h->ws + L.off_mask, h->mask_host.data(), h->mask_host.size(), cudaMemcpyHostToDevice, h->stream);
    if (e != cudaSuccess) {
      set_err(g_create_error, "clip_create: mask upload: %s", cudaGetErrorString(e));
      delete h;
      return CLIP_ECUDA;
    }
  }
  *out = h;
  return CLIP_OK;
}

int clip_init(clip_t* h, const void* d_phi0, const void* d_u0) {
  if (!h) return CLIP_EINVAL;
  if (!d_phi0 || !d_u0) { set_err(h->err, "clip_init: NULL input"); return CLIP_EINVAL; }
  if (((uintptr_t)d_phi0) % 16 || ((uintptr_t)d_u0) % 16) { set_err(h->err, "clip_init: inputs must be 16-byte aligned"); return CLIP_EINVAL; }
  if (h->overlap_open) {  // a step left open on the halo stream: order the new state after it
    cudaEventRecord(h->ev_halo, h->halo_stream);
    cudaStreamWaitEvent(h->stream, h->ev_halo, 0);
    h->overlap_open = false;
  }
  int rc = h->p.precision == 32 ? do_init<float>(h, d_phi0, d_u0) : do_init<double>(h, d_phi0, d_u0);
  if (rc == CLIP_OK) { h->inited = true; h->t = 0; }
  return rc;
}

int clip_set_u(clip_t* h, const void* d_u) {
  if (!h) return CLIP_EINVAL;
  if (!h->p.phase_only) { set_err(h->err, "clip_set_u: the handle is not in phase_only mode"); return CLIP_ESTATE; }
  if (!h->inited) { set_err(h->err, "clip_set_u: clip_init has not been called"); return CLIP_ESTATE; }
  if (!d_u || ((uintptr_t)d_u) % 16) { set_err(h->err, "clip_set_u: u must be a 16-byte aligned device pointer"); return CLIP_EINVAL; }
  const size_t bytes = 3 * (size_t)h->nx * h->ny * h->nz * h->L.word;
  cudaError_t e = cudaMemcpyAsync(h->ws + h->L.off_u, d_u, bytes, cudaMemcpyDeviceToDevice, h->stream);
  if (e != cudaSuccess) { set_err(h->err, "clip_set_u: %s", cudaGetErrorString(e)); return CLIP_ECUDA; }
  return CLIP_OK;
}

int clip_step(clip_t* h, int n) {
  if (!h) return CLIP_EINVAL;
  if (!h->inited) { set_err(h->err, "clip_step: clip_init has not been called"); return CLIP_ESTATE; }
  if (n < 0) { set_err(h->err, "clip_step: n must be >= 0"); return CLIP_EINVAL; }
  if (h->overlap_open) { set_err(h->err, "clip_step: an overlapped step is open (clip_step_halo_end missing)"); return CLIP_ESTATE; }
  return h->p.precision == 32 ? step_graphed<float>(h, n) : step_graphed<double>(h, n);
}

int clip_step_profiled(clip_t* h, int n, double* ms, long long* count) {
  if (!h) return CLIP_EINVAL;
  if (!h->inited) { set_err(h->err, "clip_step_profiled: clip_init has not been called"); return CLIP_ESTATE; }
  if (n < 0 || !ms || !count) { set_err(h->err, "clip_step_profiled: bad arguments"); return CLIP_EINVAL; }
  Prof prof;
  prof.stream = h->stream;
  int rc = h->p.precision == 32 ? do_step<float>(h, n, &prof) : do_step<double>(h, n, &prof);
  cudaError_t e = cudaStreamSynchronize(h->stream);
  if (rc == CLIP_OK && e != cudaSuccess) { set_err(h->err, "clip_step_profiled: %s", cudaGetErrorString(e)); rc = CLIP_ECUDA; }
  for (size_t k = 0; k < prof.kind.size(); ++k) {
    float t = 0.f;
    if (rc == CLIP_OK && cudaEventElapsedTime(&t, prof.ev[2 * k], prof.ev[2 * k + 1]) == cudaSuccess) {
      ms[prof.kind[k]] += t;
      count[prof.kind[k]] += 1;
    }
  }
  for (cudaEvent_t ev : prof.ev) cudaEventDestroy(ev);
  return rc;
}

int clip_kernel_kinds(void) { return KIND_COUNT; }
const char* clip_kernel_name(int kind) { return (kind >= 0 && kind < KIND_COUNT) ? KIND_NAMES[kind] : nullptr; }

int clip_get(clip_t* h, void* d_phi, void* d_p, void* d_u) {
  if (!h) return CLIP_EINVAL;
  if (!h->inited) { set_err(h->err, "clip_get: clip_init has not been called"); return CLIP_ESTATE; }
  if (((uintptr_t)d_phi) % 16 || ((uintptr_t)d_p) % 16 || ((uintptr_t)d_u) % 16) { set_err(h->err, "clip_get: outputs must be 16-byte aligned"); return CLIP_EINVAL; }
  if (!d_phi && !d_p && !d_u) return CLIP_OK;
  return h->p.precision == 32 ? do_get<float>(h, d_phi, d_p, d_u) : do_get<double>(h, d_phi, d_p, d_u);
}

int clip_destroy(clip_t* h) {
  if (!h) return CLIP_EINVAL;
  if (!h->mask_host.empty()) cudaStreamSynchronize(h->stream);  // the mask upload reads host memory we own
  if (h->ev_start) { cudaEventDestroy(h->ev_start); cudaEventDestroy(h->ev_bnd); cudaEventDestroy(h->ev_halo); }
  if (h->gexec) cudaGraphExecDestroy(h->gexec);
  delete h;
  return CLIP_OK;
}

const char* clip_last_error(const clip_t* h) { return h ? h->err : g_create_error; }

long long clip_launch_count(const clip_t* h) { return h ? h->launches : 0; }
long long clip_graph_steps(const clip_t* h) { return h ? h->graph_steps : 0; }

}  // extern "C"
