// abi.cu -- the C ABI of include/mpc_b200.h and the step scheduler of the fused SRD path.
// One CUDA stream, no host synchronisation inside mpc_step.
#include <new>

#include "internal.cuh"

using namespace mpc;

static const char* const FAMILY_NAMES[F_COUNT] = {"sweep", "cell", "collide", "scan", "scatter_slots", "rank", "gather", "memset",
                                                  "stream_key", "accum", "observables", "sweep_gather"};

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
  size_t off_A[7], off_B[7], off_key, off_slot, off_perm, off_cursor, off_offset, off_bsum, off_sums, off_lcount, off_abase, off_rec, off_obs, off_mt,
      off_tbase, off_chunk0, total;
};
// tile_cells: cells of one brick's shared-memory tile; tbase (first slot of every CTA inside every tile cell's segment,
// written by the staging sweep of a reorder) exists only where the staged reorder does: second particle copy, SRD path
Layout make_layout(bool sub, size_t n_max, size_t nkeys, size_t nbricks, size_t tile_cells, int sw, int rw, bool compact, bool generic) {
  Layout l;
  size_t o = 0;
  auto take = [&](size_t bytes) { const size_t r = o; o = align_up(o + bytes, 256); return r; };
  const size_t pn = align_up((n_max ? n_max : 1) * 4, 256);   // whole 256-byte units: consecutive arrays are contiguous
  for (int a = 0; a < 7; ++a) l.off_A[a] = take(pn);
  // the slot array sits between the two particle copies: either copy plus it = 8 contiguous arrays (the staging buffer)
  l.off_slot = take(compact ? pn * 2 : pn);
  if (compact) { l.off_B[0] = take(pn); for (int a = 1; a < 7; ++a) l.off_B[a] = l.off_B[0]; }
  else for (int a = 0; a < 7; ++a) l.off_B[a] = take(pn);
  l.off_key = take(pn);
  // (the slot array holds (id, source index) pairs, 8 bytes each, in compact mode; with the second copy present
  // those live in its first two arrays)
  l.off_perm = take(pn);
  l.off_cursor = take(nkeys * 4);
  l.off_offset = take((nkeys + 1) * 4);
  l.off_bsum = take(((nkeys + SCAN_TILE - 1) / SCAN_TILE + 1) * 4);
  l.off_sums = take(nkeys * (size_t)sw * 8);
  l.off_lcount = take(sub ? nkeys * 4 : 4);            // slab subdomain: this rank's own counts of the shared cells
  l.off_abase = take(sub ? nkeys * 4 : 4);             // ... first slot of handed-over particles inside the owner's cell segment
  l.off_rec = take(nkeys * (size_t)rw * 4);
  l.off_obs = take(OBS_HOST_DOUBLES * 8 + 256);
  l.off_mt = take(MT_TABLE * 8);
  const bool staged = !compact && !generic;
  l.off_tbase = take(staged ? nbricks * tile_cells * 4 : 4);
  // (compact SRD workspace: ranges of the previous order for the windowed gather, groups of at least an eighth of a brick)
  l.off_chunk0 = take(staged ? (nbricks + 1) * 4 : (compact && !generic) ? (8 * nbricks + 1) * 4 : 4);
  l.total = o;
  return l;
}
Layout ctx_layout(const mpc_ctx* c, size_t n_max, bool compact) {
  return make_layout(c->G.sub != 0, n_max, c->G.nkeys, c->nbricks, c->tile_bytes / (TILE_W * 4), c->G.sw, c->G.rw, compact, c->G.generic != 0);
}

void host_shift(const mpc_ctx* c, uint32_t t, float s[3]) {
  s[0] = s[1] = s[2] = 0.0f;
  if (!c->p.grid_shift) return;
  const Block4 o = philox(0u, 0u, t, TAG_SHIFT, c->G.k0, c->G.k1);
  s[0] = (u01_co(o.a) - 0.5f) * c->G.a;
  s[1] = (u01_co(o.b) - 0.5f) * c->G.a;
  s[2] = (u01_co(o.c) - 0.5f) * c->G.a;
}

// Lees-Edwards displacement of the image above at the time the positions of step t refer to, (t + 1) h (U21)
float host_le_offset(const mpc_ctx* c, uint32_t t) {
  if (c->p.shear_rate == 0.0f) return 0.0f;
  const double Ud = (double)c->p.shear_rate * (double)c->G.L[2];
  double d = fmod(Ud * (double)c->p.dt * ((double)t + 1.0), (double)c->G.L[0]);
  if (d < 0.0) d += (double)c->G.L[0];
  return (float)d;
}

// SRD: step t = sweep (collision of t-1 if one is pending + MOVE of t + sums of t), [reorder], PROCESS_CELLS of t.
// The collision of the last step stays pending: the next call's first sweep applies it (flush_collide otherwise).
// phase: 0 = whole steps; slab subdomains run ONE step in two calls around the barrier of the ranks: 1 = the sweep,
// 2 = PROCESS_CELLS and the local reorder (mpc_sub_begin / mpc_sub_end)
int steps_srd(mpc_ctx* c, int nsteps, int phase = 0) {
  Geo& G = c->G;
  const size_t n = c->n;                           // (slab subdomains: c->n changes when a folded reorder completes; one step per call there)
  float sp[3] = {G.s[0], G.s[1], G.s[2]};          // shift of the pending step (if any)
  for (int k = 0; k < nsteps; ++k) {
    const bool rebin = (c->t % (uint32_t)c->p.rebin_every) == 0u;
    // reorder folded into this sweep (rank pass) and the next two (scatter into the new order through 32-byte staging
    // records, read back): needs two more steps in this call, the order of the last reorder, the second particle copy,
    // and rebin_every >= 3
    // (slab subdomains: the caller promises the further steps in mpc_sub_begin; the folded reorder there also hands the
    // particles of the halo layers over to their new owners)
    // (a slab rank decides from what ALL ranks share: the step, the promised steps, the debug flags, and staging buffers that
    // either every rank has or none (mpc_sub_connect). Not from its own particle count: an empty slab takes part, it may be
    // handed particles)
    bool stage = rebin && c->reorder_stage == 0 && c->have_order && c->tbase && !c->compact && (n != 0 || G.sub) &&
                 !(c->debug & (MPC_DEBUG_NO_FUSE_GATHER | MPC_DEBUG_EAGER_CANONICAL | MPC_DEBUG_ATOMIC_SCATTER)) &&
                 (phase == 0 ? k + 2 < nsteps : c->sub_ahead >= 2) && c->p.rebin_every >= 3;
    if (phase == 1) c->sub_stage = stage;
    if (phase == 2) stage = c->sub_stage;
    if (phase != 2) {
      G.t = c->t;
      host_shift(c, c->t, G.s);
      c->le_dprev = G.le_d;
      G.le_d = host_le_offset(c, c->t);
      if (!c->sums_clean) { FamilyTimer ft(c, F_MEMSET); CU(cudaMemsetAsync(c->sums, 0, (size_t)G.nkeys * G.sw * 8, c->stream)); }
      c->sums_clean = false;
      // the new order holds the particles that have arrived, not those that have left (count read in mpc_sub_end of the reorder step)
      if (G.sub && c->reorder_stage == 2) c->n = c->sub_nn;
      {
        const int io = c->reorder_stage == 1 ? IO_SCATTER : c->reorder_stage == 2 ? IO_AOS_IN : (stage ? IO_RANK : IO_PLAIN);
        if (c->n) {
          FamilyTimer ft(c, io != IO_PLAIN ? F_SWEEPG : F_SWEEP);
          const int rc = launch_sweep(c, c->collide_pending, rebin && !stage, io, sp);
          if (rc) return rc;
        }
        if (io == IO_SCATTER) c->reorder_stage = 2;      // (also on a slab rank without particles: its neighbours' passes go on)
        else if (io == IO_AOS_IN) c->reorder_stage = 0;
      }
      if (phase == 1) return MPC_OK;
    }
    // all but the last step of the call: k_cell clears the sums it has read (the last step's stay for
    // mpc_observables / mpc_get_cells). Slab subdomains always clear: the neighbours add into these sums in the next sweep
    const int zero = (k + 1 < nsteps || phase == 2) ? 1 : 0;
    // a folded reorder scans compact counts that k_cell writes while it reads the sums anyway (the scan would otherwise
    // read every cell's 24 bytes twice); the other reorders read the counts from the sums, before k_cell clears them
    // (slab subdomains: always the compact counts: the sums of shared cells include the neighbours' particles)
    const bool compact_counts = stage || G.sub;
    if (rebin && !compact_counts && n) {
      const int rc = do_reorder(c, false, (c->debug & MPC_DEBUG_EAGER_CANONICAL) != 0, false);
      if (rc) return rc;
    }
    {   // (a slab subdomain without particles still has cells: its neighbours' particles in the shared layers)
      FamilyTimer ft(c, F_CELL);
      const int rc = (n || G.sub) ? launch_cell(c, zero, (rebin && compact_counts) ? c->cursor : nullptr, G.sub && stage) : MPC_OK;
      if (rc) return rc;
    }
    if (rebin && compact_counts && (n || G.sub)) {
      const int rc = do_reorder(c, stage, false, true);
      if (rc) return rc;
      if (G.sub && stage) {
        // Hand-over: the scan's total is this rank's particle count in the new order (own particles that stay + arrivals).
        // It is checked HERE, before the barrier that ends the step: in the next step this rank and both neighbours write
        // 32-byte records at slots up to that total into this rank's staging buffer, which holds n_max of them. Too many:
        // the context is dead (sticky), and the caller must stop every rank before the next mpc_sub_begin.
        uint32_t nn = 0;
        CU(cudaMemcpyAsync(&nn, c->offset + G.nkeys, 4, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        if (nn > c->n_max) {
          c->sticky = true;
          return fail(c, MPC_ENOMEM, "slab subdomain: the reorder would hand this rank more particles than n_max holds; no rank may start the next step");
        }
        c->sub_nn = nn;
      }
    }
    if (n || G.sub) {
      c->sums_clean = zero != 0;
      c->collide_pending = n != 0 || G.sub;   // (slab rank: particles handed to an empty slab arrive with this collision still to apply)
    }
    sp[0] = G.s[0]; sp[1] = G.s[1]; sp[2] = G.s[2];
    c->t++;
    c->have_cells = true;
  }
  if (c->debug & MPC_DEBUG_EAGER_COLLIDE) return flush_collide(c);
  return MPC_OK;
}

int set_state_impl(mpc_ctx* c, unsigned long long n, const float* const src[6], const unsigned* id, unsigned step,
                   cudaMemcpyKind kind) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->bound) return fail(c, MPC_ESTATE, "mpc_set_state before mpc_bind");
  if (n > c->n_max) return fail(c, MPC_ENOMEM, "n exceeds the n_max given to mpc_bind");
  for (int a = 0; a < 6; ++a) if (n && !src[a]) return fail(c, MPC_EINVAL, "NULL state array");
  // a slab rank in the middle of a step or of a folded reorder: its neighbours are writing (or about to write) particles into its staging buffer
  if (c->G.sub && (c->reorder_stage || c->sub_open))
    return fail(c, MPC_ESTATE, "slab subdomain: mpc_set_state between mpc_sub_begin and mpc_sub_end or while a folded reorder is in flight");
  CU(cudaSetDevice(c->device));
  for (int a = 0; a < 6; ++a)
    if (n) CU(cudaMemcpyAsync(c->A[a], src[a], n * 4, kind, c->stream));
  if (n) {
    if (id) CU(cudaMemcpyAsync(c->A[6], id, n * 4, kind, c->stream));
    else { const int rc = launch_iota(c); if (rc) return rc; }    // ids 0..n_max-1
  }
  CU(cudaMemsetAsync(c->nrange, 0, 8, c->stream));
  c->n = n; c->t = step; c->have_state = true; c->have_cells = false; c->have_order = false; c->reorder_stage = 0; c->sub_open = false;
  c->order_canonical = true; c->order_spread = 0; c->collide_pending = false;
  return MPC_OK;
}
int get_state_impl(mpc_ctx* c, float* const dst[6], unsigned* id, cudaMemcpyKind kind) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->have_state) return fail(c, MPC_ESTATE, "mpc_get_state before mpc_set_state");
  if (c->reorder_stage) return fail(c, MPC_ESTATE, "slab subdomain: a folded reorder is in flight (run the steps promised to mpc_sub_begin first)");
  CU(cudaSetDevice(c->device));
  { const int rc = flush_collide(c); if (rc) return rc; }
  { const int rc = canonicalise(c); if (rc) return rc; }
  for (int a = 0; a < 6; ++a)
    if (dst[a] && c->n) CU(cudaMemcpyAsync(dst[a], c->A[a], c->n * 4, kind, c->stream));
  if (id && c->n) CU(cudaMemcpyAsync(id, c->A[6], c->n * 4, kind, c->stream));
  if (kind == cudaMemcpyDeviceToHost) CU(cudaStreamSynchronize(c->stream));
  return MPC_OK;
}

}  // namespace

// apply the pending collision of the last step (SRD path): velocities become those of the fully collided state
int flush_collide(mpc_ctx* c) {
  if (!c->collide_pending || c->n == 0) { c->collide_pending = false; return MPC_OK; }
  FamilyTimer ft(c, F_COLLIDE);
  const int rc = launch_collide_pos(c);
  if (rc == MPC_OK) c->collide_pending = false;
  return rc;
}

extern "C" {

int mpc_create(mpc_ctx** out, const float box[3], const int cells[3], float n_per_cell, const mpc_params* p,
               unsigned long long seed) {
  if (!out) return MPC_EINVAL;
  *out = nullptr;
  if (!box || !cells || !p) return MPC_EINVAL;
  // >= 3 cells per axis: with fewer, a particle shares a collision cell with its own periodic image
  for (int d = 0; d < 3; ++d) if (cells[d] < 3 || !(box[d] > 0.0f)) return MPC_EINVAL;
  const float a = box[0] / (float)cells[0];
  for (int d = 1; d < 3; ++d) if (box[d] / (float)cells[d] != a) return MPC_EINVAL;
  if (p->collision < 0 || p->collision > 1) return MPC_EINVAL;
  if (!(p->dt > 0.0f) || !(p->kT > 0.0f) || !(p->mass > 0.0f) || p->rebin_every < 1 || !(n_per_cell > 0.0f)) return MPC_EINVAL;
  size_t tile_cells = 1;
  for (int d = 0; d < 3; ++d) {
    const int b = p->brick[d];
    if (b < 1 || (b & (b - 1)) != 0 || b > 64) return MPC_EINVAL;   // powers of two
    tile_cells *= (size_t)(b + 2 * HALO);
  }
  if (tile_cells * TILE_W * 4 > MAX_TILE_BYTES) return MPC_EINVAL;
  int nwall = 0, wall = -1;
  for (int d = 0; d < 3; ++d) {
    if (p->bc[d] < 0 || p->bc[d] > 2) return MPC_EINVAL;
    if (p->bc[d] != 0) { nwall++; wall = d; if (p->g[d] != 0.0f) return MPC_EINVAL; }
  }
  if (nwall > 1) return MPC_EINVAL;
  if (nwall && (p->conserve_L || p->collision == 1) && !p->phantoms) return MPC_EINVAL;     // needs explicit phantoms (U8, U22)
  if (p->phantoms < 0 || p->phantoms > 1 || (p->phantoms && (!nwall || p->bc[wall] != 1))) return MPC_EINVAL;
  if (p->solute_mass < 0.0f) return MPC_EINVAL;
  if ((p->phantoms || p->solute_mass > 0.0f) && (p->rebin_every != 1 || p->shear_rate != 0.0f)) return MPC_EINVAL;   // per-cell segment pass only
  if (p->wall_velocity != 0.0f && (!nwall || wall == 0 || p->bc[wall] != 1)) return MPC_EINVAL;    // moving walls: no-slip, flow along x (U24)
  if (p->collision == 0 && p->conserve_L && p->thermostat) return MPC_EINVAL;
  if (p->collision == 1 && p->rebin_every != 1) return MPC_EINVAL;
  if (p->shear_rate != 0.0f && (nwall || p->collision == 1 || p->conserve_L)) return MPC_EINVAL;   // Lees-Edwards: periodic SRD only (U21)
  const bool sub = p->sub_nz != 0 || p->sub_z0 != 0;
  if (sub) {   // slab subdomain: periodic SRD -a without force, whole brick layers, one brick layer of halo
    const int bz = p->brick[2];
    if (nwall || p->collision != 0 || p->conserve_L || p->shear_rate != 0.0f || p->phantoms || p->solute_mass > 0.0f) return MPC_EINVAL;
    if (p->g[0] != 0.0f || p->g[1] != 0.0f || p->g[2] != 0.0f) return MPC_EINVAL;
    if (p->sub_z0 < 0 || p->sub_z0 >= cells[2] || p->sub_z0 % bz || p->sub_nz % bz || p->sub_nz < 2 * bz || p->sub_nz + 2 * bz > cells[2]) return MPC_EINVAL;
  }
  mpc_ctx* c = new (std::nothrow) mpc_ctx();   // value-initialised: all zero
  if (!c) return MPC_ENOMEM;
  c->p = *p; c->seed = seed;
  c->hbuf = new (std::nothrow) double[OBS_HOST_DOUBLES];
  if (!c->hbuf) { delete c; return MPC_ENOMEM; }
  Geo& G = c->G;
  G.a = a; G.inv_a = 1.0f / a; G.wall = wall; G.slip = (wall >= 0 && p->bc[wall] == 2) ? 1 : 0;
  unsigned long long nk = 1, nbr = 1;
  for (int d = 0; d < 3; ++d) {
    int bs = 0;
    while ((1 << bs) < p->brick[d]) ++bs;
    G.bs[d] = bs;
    G.L[d] = box[d]; G.n[d] = cells[d]; G.bc[d] = p->bc[d]; G.g[d] = p->g[d];
    G.m[d] = cells[d] + (p->bc[d] != 0 ? 2 : 0);
    if (sub && d == 2) G.m[d] = p->sub_nz + 2 * p->brick[2];    // local layers: own + one brick layer of halo on either side
    G.mb[d] = (G.m[d] + p->brick[d] - 1) >> bs;
    nk *= (unsigned long long)G.mb[d] << bs;
    nbr *= (unsigned long long)G.mb[d];
  }
  if (nk >= 0xffffffffull) { delete[] c->hbuf; delete c; return MPC_EINVAL; }
  G.nkeys = (uint32_t)nk;
  c->nbricks = (uint32_t)nbr;
  c->tile_bytes = tile_cells * TILE_W * 4;
  c->three_ctas = 3 * (c->tile_bytes + 1024) <= 227 * 1024;
  c->fast_brick = (G.bs[0] == 4 && G.bs[1] == 4 && G.bs[2] == 3);
  c->pow2_cells = wall < 0 && !(G.m[0] & (G.m[0] - 1)) && !(G.m[1] & (G.m[1] - 1)) && (sub || !(G.m[2] & (G.m[2] - 1)));
  if (sub) { G.sub = 1; G.nzg = cells[2]; G.zoff = p->sub_z0 - p->brick[2]; G.nbz = G.mb[2]; }
  {
    const int bvs = G.bs[0] + G.bs[1] + G.bs[2];
    c->cell_cpb_shift = bvs > 8 ? bvs - 8 : 0;      // k_cell: CTAs of 256 cells
    c->cell_grid = dim3((unsigned)G.mb[0] << c->cell_cpb_shift, (unsigned)G.mb[1], (unsigned)G.mb[2]);
    c->seg_cpb_shift = bvs > 7 ? bvs - 7 : 0;       // per-cell kernels of the generic path: CTAs of 128 cells
    c->seg_grid = dim3((unsigned)G.mb[0] << c->seg_cpb_shift, (unsigned)G.mb[1], (unsigned)G.mb[2]);
    if (G.mb[1] > 65535 || G.mb[2] > 65535) { delete[] c->hbuf; delete c; return MPC_EINVAL; }
  }
  G.dt = p->dt; G.kT = p->kT; G.mass = p->mass;
  G.sigma = (float)sqrt((double)p->kT / (double)p->mass);
  G.cosa = (float)cos((double)p->alpha); G.sina = (float)sin((double)p->alpha);
  G.k0 = (uint32_t)(seed & 0xffffffffull); G.k1 = (uint32_t)(seed >> 32);
  philox_round_keys(G.k0, G.k1, G.rk);
  G.nbar = (int)lround((double)n_per_cell);
  const int ue = (int)lround(log2((double)G.sigma));        // thermal velocity rounded to a power of two
  G.fxv = (float)ldexp(1.0, 22 - ue); G.fxv_inv = ldexp(1.0, ue - 22);
  G.fxe = (float)ldexp(1.0, 22 - 2 * ue); G.fxe_inv = ldexp(1.0, 2 * ue - 22);
  G.vmax = (float)ldexp(1.0, ue + 3);
  G.shear = p->shear_rate != 0.0f ? 1 : 0;
  G.le_u = (float)((double)p->shear_rate * (double)box[2]);
  G.le_d = 0.0f;
  G.collision = p->collision; G.thermostat = p->thermostat; G.conserve_L = p->conserve_L;
  G.phantoms = p->phantoms; G.solute_id0 = p->solute_id0; G.solute_mass = p->solute_mass; G.wall_u = p->wall_velocity;
  G.generic = (p->collision == 1 || p->conserve_L || p->phantoms || p->solute_mass > 0.0f) ? 1 : 0;
  G.sw = (p->collision == 0 && p->conserve_L) ? 16 : 3;
  G.rw = p->conserve_L ? 16 : REC_W;
  *out = c;
  return MPC_OK;
}

int mpc_num_keys(const mpc_ctx* c, unsigned long long* nkeys) {
  if (!c || !nkeys) return MPC_EINVAL;
  *nkeys = c->G.nkeys;
  return MPC_OK;
}

int mpc_num_particles(const mpc_ctx* c, unsigned long long* n) {
  if (!c || !n) return MPC_EINVAL;
  *n = c->n;
  return MPC_OK;
}

int mpc_workspace_bytes(const mpc_ctx* c, unsigned long long n_max, int compact, size_t* bytes) {
  if (!c || !bytes || n_max > 0xffffffffull) return MPC_EINVAL;
  *bytes = ctx_layout(c, (size_t)n_max, compact != 0).total;
  return MPC_OK;
}

int mpc_bind(mpc_ctx* c, void* workspace, size_t bytes, unsigned long long n_max, void* cuda_stream) {
  if (!c) return MPC_EINVAL;
  if (!workspace || ((uintptr_t)workspace & 255u) || n_max > 0xffffffffull) return fail(c, MPC_EINVAL, "workspace NULL, misaligned or n_max too large");
  {
    cudaPointerAttributes at;
    int cur = -1;
    CU(cudaGetDevice(&cur));
    CU(cudaPointerGetAttributes(&at, workspace));
    if (at.type != cudaMemoryTypeDevice) return fail(c, MPC_EINVAL, "workspace is not device memory");
    if (at.device != cur) return fail(c, MPC_EINVAL, "workspace lives on another device than the current one");
    c->device = cur;
  }
  Layout l = ctx_layout(c, (size_t)n_max, false);
  bool compact = false;
  if (bytes < l.total) { l = ctx_layout(c, (size_t)n_max, true); compact = true; }
  if (bytes < l.total) return fail(c, MPC_ENOMEM, "workspace smaller than mpc_workspace_bytes(n_max, compact=1)");
  c->ws = (char*)workspace; c->ws_bytes = bytes; c->n_max = (size_t)n_max; c->compact = compact;
  c->stream = (cudaStream_t)cuda_stream;
  for (int a = 0; a < 7; ++a) { c->A[a] = (uint32_t*)(c->ws + l.off_A[a]); c->Bf[a] = (uint32_t*)(c->ws + l.off_B[a]); }
  c->key = (uint32_t*)(c->ws + l.off_key);
  c->slot_id = (uint32_t*)(c->ws + l.off_slot); c->perm = (uint32_t*)(c->ws + l.off_perm);
  c->cursor = (uint32_t*)(c->ws + l.off_cursor); c->offset = (uint32_t*)(c->ws + l.off_offset);
  c->bsum = (uint32_t*)(c->ws + l.off_bsum);
  c->sums = (u64*)(c->ws + l.off_sums); c->rec = (float*)(c->ws + l.off_rec); c->obs = (double*)(c->ws + l.off_obs);
  c->nsing = (u64*)(c->ws + l.off_obs + OBS_HOST_DOUBLES * 8);
  c->nrange = c->nsing + 1;
  c->G.nrange = c->nrange;
  c->G.lcount = c->G.sub ? (uint32_t*)(c->ws + l.off_lcount) : nullptr;
  c->G.abase = c->G.sub ? (uint32_t*)(c->ws + l.off_abase) : nullptr;
  c->G.peer[0] = c->G.peer[1] = nullptr;
  {   // table of the thermostat draw (cell.cuh)
    fill_mt_table(c->mt_host);
    CU(cudaMemcpyAsync(c->ws + l.off_mt, c->mt_host, MT_TABLE * 8, cudaMemcpyHostToDevice, c->stream));
    c->G.mt_c = (const float*)(c->ws + l.off_mt);
  }
  const bool staged = !compact && !c->G.generic;
  c->tbase = staged ? (uint32_t*)(c->ws + l.off_tbase) : nullptr;
  c->chunk0 = (staged || (compact && !c->G.generic)) ? (uint32_t*)(c->ws + l.off_chunk0) : nullptr;
  c->gwin_shift = 0; c->gwin_cap = 0;
  if (compact && !c->G.generic) {
    // window of k_gather_win: the largest aligned part of a brick (down to an eighth, at least 32 keys: the lane-spread order
    // permutes inside groups of 32) whose mean particle number, plus 20 %, fits in 100 KB, so that two CTAs share an SM
    const int bvs = c->G.bs[0] + c->G.bs[1] + c->G.bs[2];
    for (int sh = bvs; sh >= bvs - 3 && sh >= SPREAD_GROUP_SHIFT; --sh) {
      const double elems = 1.2 * (double)(1u << sh) * (double)c->G.nbar + 256.0;
      if (elems * 4.0 <= 100.0 * 1024.0) { c->gwin_shift = sh; c->gwin_cap = (uint32_t)elems; break; }
    }
  }
  CU(cudaMemsetAsync(c->nrange, 0, 8, c->stream));
  c->bound = true; c->have_state = false; c->have_cells = false; c->have_order = false; c->sums_clean = false; c->reorder_stage = 0;
  c->collide_pending = false; c->order_spread = 0; c->n = 0;
  if (c->tile_bytes > 48 * 1024) {
    const cudaError_t e = sweep_set_attributes(c->tile_bytes);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaFuncSetAttribute(k_sweep, MaxDynamicSharedMemorySize)");
  }
  return MPC_OK;
}

int mpc_set_debug(mpc_ctx* c, unsigned flags) {
  if (!c) return MPC_EINVAL;
  if (flags & ~(MPC_DEBUG_NO_FUSE_GATHER | MPC_DEBUG_EAGER_CANONICAL | MPC_DEBUG_ATOMIC_SCATTER | MPC_DEBUG_EAGER_COLLIDE | MPC_DEBUG_NO_LANE_SPREAD)) return fail(c, MPC_EINVAL, "unknown debug flag");
  if (c->reorder_stage) return fail(c, MPC_ESTATE, "internal: reorder in flight");   // cannot happen between API calls
  c->debug = flags;
  return MPC_OK;
}

int mpc_set_state(mpc_ctx* c, unsigned long long n, const float* x, const float* y, const float* z, const float* vx,
                  const float* vy, const float* vz, const unsigned* id, unsigned step) {
  const float* const src[6] = {x, y, z, vx, vy, vz};
  return set_state_impl(c, n, src, id, step, cudaMemcpyDeviceToDevice);
}
int mpc_set_state_host(mpc_ctx* c, unsigned long long n, const float* x, const float* y, const float* z, const float* vx,
                       const float* vy, const float* vz, const unsigned* id, unsigned step) {
  const float* const src[6] = {x, y, z, vx, vy, vz};
  return set_state_impl(c, n, src, id, step, cudaMemcpyHostToDevice);
}

int mpc_step(mpc_ctx* c, int nsteps) {
  if (!c || nsteps < 0) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->bound || !c->have_state) return fail(c, MPC_ESTATE, "mpc_step before mpc_bind / mpc_set_state");
  if (c->G.sub) return fail(c, MPC_ESTATE, "slab subdomain: use mpc_sub_begin / mpc_sub_end around the barrier of the ranks");
  CU(cudaSetDevice(c->device));
  return c->G.generic ? steps_generic(c, nsteps) : steps_srd(c, nsteps);
}

int mpc_sub_export(mpc_ctx* c, void* device_ptrs[3], int* brick_layers) {
  if (!c || !device_ptrs || !brick_layers) return MPC_EINVAL;
  if (!c->G.sub) return fail(c, MPC_ESTATE, "not a slab subdomain");
  if (!c->bound) return fail(c, MPC_ESTATE, "mpc_sub_export before mpc_bind");
  device_ptrs[0] = c->sums; device_ptrs[1] = c->offset; device_ptrs[2] = c->compact ? nullptr : aos_base(c);
  *brick_layers = c->G.nbz;
  return MPC_OK;
}

int mpc_sub_connect(mpc_ctx* c, void* const below[3], int brick_layers_below, void* const above[3], int brick_layers_above) {
  if (!c || !below || !above || !below[0] || !above[0] || !below[1] || !above[1] || brick_layers_below < 4 || brick_layers_above < 4) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->G.sub) return fail(c, MPC_ESTATE, "not a slab subdomain");
  if (!c->bound) return fail(c, MPC_ESTATE, "mpc_sub_connect before mpc_bind");
  CU(cudaSetDevice(c->device));
  Geo& G = c->G;
  const long long layer_keys = ((long long)G.mb[0] * G.mb[1]) << (G.bs[0] + G.bs[1] + G.bs[2]);   // keys of one brick layer
  G.peer_koff[0] = (long long)(brick_layers_below - 2) * layer_keys;   // my layers 0, 1 = its last two
  G.peer_koff[1] = -(long long)(G.nbz - 2) * layer_keys;               // my last two = its layers 0, 1
  void* const* side[2] = {below, above};
  for (int d = 0; d < 2; ++d) {
    G.peer[d] = (u64*)side[d][0]; G.peer_offset[d] = (const uint32_t*)side[d][1]; G.peer_aos[d] = (float*)side[d][2];
  }
  if (!G.peer_aos[0] || !G.peer_aos[1] || c->compact) c->tbase = nullptr;   // no staging buffers: local reorders stay unfolded, hand-over by mpc_sub_pack
  const int rc = launch_sub_clear(c);
  if (rc) return rc;
  c->sums_clean = true;
  return MPC_OK;
}

static int sub_phase(mpc_ctx* c, int phase, int steps_ahead) {
  if (!c || steps_ahead < 0) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->G.sub) return fail(c, MPC_ESTATE, "not a slab subdomain");
  if (!c->bound || !c->have_state || !c->G.peer[0]) return fail(c, MPC_ESTATE, "slab subdomain: needs mpc_bind, mpc_sub_connect and mpc_set_state first");
  if ((phase == 1) == c->sub_open) return fail(c, MPC_ESTATE, "mpc_sub_begin and mpc_sub_end must alternate");
  CU(cudaSetDevice(c->device));
  if (phase == 1) c->sub_ahead = steps_ahead;
  const int rc = steps_srd(c, 1, phase);
  if (rc == MPC_OK) c->sub_open = (phase == 1);
  return rc;
}
int mpc_sub_pack(mpc_ctx* c, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id, unsigned long long counts[3]) {
  if (!c || !x || !y || !z || !vx || !vy || !vz || !id || !counts) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->G.sub) return fail(c, MPC_ESTATE, "not a slab subdomain");
  if (!c->have_state || c->sub_open || c->reorder_stage) return fail(c, MPC_ESTATE, "mpc_sub_pack needs a state, no open step and no reorder in flight");
  CU(cudaSetDevice(c->device));
  { const int rc = flush_collide(c); if (rc) return rc; }
  float* const out[6] = {x, y, z, vx, vy, vz};
  return sub_pack_impl(c, out, id, counts);
}
int mpc_sub_begin(mpc_ctx* c, int steps_ahead) { return sub_phase(c, 1, steps_ahead); }
int mpc_sub_end(mpc_ctx* c) { return sub_phase(c, 2, 0); }

int mpc_get_state(mpc_ctx* c, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id) {
  float* const dst[6] = {x, y, z, vx, vy, vz};
  return get_state_impl(c, dst, id, cudaMemcpyDeviceToDevice);
}
int mpc_get_state_host(mpc_ctx* c, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id) {
  float* const dst[6] = {x, y, z, vx, vy, vz};
  return get_state_impl(c, dst, id, cudaMemcpyDeviceToHost);
}

int mpc_observables(mpc_ctx* c, mpc_obs* out, float* profile_host, int n_profile) {
  if (!c || !out) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->have_state) return fail(c, MPC_ESTATE, "mpc_observables before mpc_set_state");
  if (c->reorder_stage) return fail(c, MPC_ESTATE, "slab subdomain: a folded reorder is in flight (run the steps promised to mpc_sub_begin first)");
  CU(cudaSetDevice(c->device));
  { const int rc = flush_collide(c); if (rc) return rc; }
  return observables_impl(c, out, profile_host, n_profile);
}

int mpc_get_cells(mpc_ctx* c, unsigned* count, float* px, float* py, float* pz, float* e2, unsigned* key) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->have_cells) return fail(c, MPC_ESTATE, "mpc_get_cells before the first mpc_step");
  CU(cudaSetDevice(c->device));
  return get_cells_impl(c, count, px, py, pz, e2, key);
}

void mpc_philox4x32_10(const unsigned ctr[4], const unsigned key[2], unsigned out[4]) {
  const Block4 o = philox(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1]);
  out[0] = o.a; out[1] = o.b; out[2] = o.c; out[3] = o.d;
}

unsigned long long mpc_launch_count(const mpc_ctx* c) { return c ? c->launches : 0ull; }

int mpc_profile_enable(mpc_ctx* c, int on) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (on && !c->prof_ev) {
    c->prof_ev = new (std::nothrow) cudaEvent_t[2 * PROF_MAX_PAIRS];
    c->prof_fam = new (std::nothrow) int[PROF_MAX_PAIRS];
    if (!c->prof_ev || !c->prof_fam) return fail(c, MPC_ENOMEM, "profile buffers");
    for (int i = 0; i < 2 * PROF_MAX_PAIRS; ++i) CU(cudaEventCreate(&c->prof_ev[i]));
  }
  c->prof_on = on != 0;
  return MPC_OK;
}

int mpc_profile_read(mpc_ctx* c, int* n_families, const char** names, double* total_ms, unsigned long long* launches) {
  if (!c || !n_families) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (c->prof_pairs) CU(cudaStreamSynchronize(c->stream));
  for (int i = 0; i < c->prof_pairs; ++i) {
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
    c->prof_ms[c->prof_fam[i]] += ms;
  }
  c->prof_pairs = 0;
  *n_families = F_COUNT;
  for (int f = 0; f < F_COUNT; ++f) {
    if (names) names[f] = FAMILY_NAMES[f];
    if (total_ms) total_ms[f] = c->prof_ms[f];
    if (launches) launches[f] = c->prof_launches[f];
    c->prof_ms[f] = 0.0; c->prof_launches[f] = 0;
  }
  return MPC_OK;
}

const char* mpc_last_error(const mpc_ctx* c) { return c ? c->err : "null context"; }

int mpc_destroy(mpc_ctx* c) {
  if (c) {
    delete[] c->hbuf;
    if (c->prof_ev) for (int i = 0; i < 2 * PROF_MAX_PAIRS; ++i) cudaEventDestroy(c->prof_ev[i]);
    delete[] c->prof_ev;
    delete[] c->prof_fam;
  }
  delete c;
  return MPC_OK;
}

}  // extern "C"
