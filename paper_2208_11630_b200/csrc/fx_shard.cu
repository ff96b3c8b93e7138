// fx_shard.cu -- multi-GPU sharding of a block batch [SURVEY.md 8(e); MPI between ranks, L69: blocks are
// independent within a stage once the Grid unit has resolved their boundaries].
//
// One process per GPU.  Rank r owns a contiguous run of the block order (a Morton run when the global table was built
// with FX_ORDER_MORTON) and keeps, behind its owned blocks, one GHOST block for every block of another rank that an
// owned block names as a neighbour.  A ghost block is a read-only source of halo cells: the stage kernels advance the
// owned blocks only (FX_OPT_OWNED_BLOCKS) and read a ghost exactly as they read any neighbour's interior, so no kernel
// changes.  Before every stage the R-deep face slabs of the stage input that face a cut are packed, exchanged (the
// binding hands the packed buffers to torch.distributed / NCCL over NVLink) and unpacked into the ghosts' interiors:
// 16 x 16 x 2 x 5 x 8 B = 20 480 B per cut face for PLM, 30 720 B for WENO5 -- about 2 % of a rank's stage traffic at
// config-5 scale.  The time step is the minimum over the ranks' own reductions (one 8-byte all-reduce per step).
//
// This file: the host-side partitioner (pure index logic, no GPU needed: tested with 2 gloo ranks on the CPU against
// the single-domain oracle) and the two device kernels that pack and unpack face slabs.
#include <algorithm>
#include <map>
#include <new>
#include <vector>

#include "fx_internal.h"

struct fx_shard {
  long long nglobal;
  int nranks, rank;
  long long begin, end;                 // owned global ids [begin, end)
  std::vector<long long> ghosts;        // global ids of the ghost blocks, ascending
  std::vector<int32_t> neigh_local;     // [(owned + ghosts)][6]
  std::vector<int32_t> send_items, recv_items;  // [n][2]: local block id, side (0..5); grouped by peer, each group sorted by (global id, side)
  std::vector<long long> send_counts, recv_counts;  // items per peer
};

static inline long long fx_run_begin(long long n, int nranks, int r) { return n * (long long)r / nranks; }
static inline int fx_owner(long long g, long long n, int nranks) {
  int r = (int)((g * nranks) / n);  // first guess, then correct (integer division of the run bounds)
  while (r > 0 && g < fx_run_begin(n, nranks, r)) --r;
  while (r + 1 < nranks && g >= fx_run_begin(n, nranks, r + 1)) ++r;
  return r;
}

extern "C" int fx_shard_create(fx_shard **out, int64_t nblocks_global, const int32_t *neigh, int nranks, int rank) {
  if (!out) return fx_fail(FX_ERR_INVALID_ARG, "shard_create: null output");
  *out = nullptr;
  if (nblocks_global < 1 || !neigh || nranks < 1 || rank < 0 || rank >= nranks || nranks > nblocks_global)
    return fx_fail(FX_ERR_INVALID_ARG, "shard_create: need 1 <= nranks <= nblocks, 0 <= rank < nranks and a table");
  for (long long i = 0; i < nblocks_global * 6; ++i)
    if (neigh[i] >= nblocks_global) return fx_fail(FX_ERR_INVALID_ARG, "shard_create: neighbour id %d out of range", neigh[i]);
  fx_shard *s = new (std::nothrow) fx_shard();
  if (!s) return fx_fail(FX_ERR_INVALID_ARG, "shard_create: out of host memory");
  const long long N = nblocks_global;
  s->nglobal = N;
  s->nranks = nranks;
  s->rank = rank;
  s->begin = fx_run_begin(N, nranks, rank);
  s->end = fx_run_begin(N, nranks, rank + 1);
  // what rank q needs from rank p: the slab of G on side f^1 for every owned B of q whose face f names a block G of p
  // (the kernels read a +x neighbour's first R columns, a -x neighbour's last R, and so on).  Every rank derives every
  // pair's list from the global table, so sender and receiver agree on content and order without talking.
  auto items_for = [&](int q, std::vector<std::vector<std::pair<long long, int>>> &per_src) {
    per_src.assign(nranks, {});
    const long long b0 = fx_run_begin(N, nranks, q), b1 = fx_run_begin(N, nranks, q + 1);
    for (long long B = b0; B < b1; ++B)
      for (int f = 0; f < 6; ++f) {
        const long long G = neigh[B * 6 + f];
        if (G < 0) continue;
        const int p = fx_owner(G, N, nranks);
        if (p != q) per_src[p].push_back({G, f ^ 1});
      }
    for (auto &v : per_src) {
      std::sort(v.begin(), v.end());
      v.erase(std::unique(v.begin(), v.end()), v.end());
    }
  };
  std::vector<std::vector<std::pair<long long, int>>> mine;
  items_for(rank, mine);
  for (auto &v : mine)
    for (auto &it : v) s->ghosts.push_back(it.first);
  std::sort(s->ghosts.begin(), s->ghosts.end());
  s->ghosts.erase(std::unique(s->ghosts.begin(), s->ghosts.end()), s->ghosts.end());
  const long long nown = s->end - s->begin, nloc = nown + (long long)s->ghosts.size();
  if (nloc > 2147483647LL) {
    delete s;
    return fx_fail(FX_ERR_INVALID_ARG, "shard_create: too many local blocks");
  }
  auto local_of = [&](long long g) -> int32_t {
    if (g >= s->begin && g < s->end) return (int32_t)(g - s->begin);
    return (int32_t)(nown + (std::lower_bound(s->ghosts.begin(), s->ghosts.end(), g) - s->ghosts.begin()));
  };
  s->neigh_local.assign((size_t)nloc * 6, FX_BC_OUTFLOW);  // a ghost's own faces are never resolved by a stage kernel
  for (long long B = s->begin; B < s->end; ++B)
    for (int f = 0; f < 6; ++f) {
      const int32_t v = neigh[B * 6 + f];
      s->neigh_local[(size_t)(B - s->begin) * 6 + f] = v >= 0 ? local_of(v) : v;
    }
  s->recv_counts.assign(nranks, 0);
  s->send_counts.assign(nranks, 0);
  for (int p = 0; p < nranks; ++p) {
    s->recv_counts[p] = (long long)mine[p].size();
    for (auto &it : mine[p]) {
      s->recv_items.push_back(local_of(it.first));
      s->recv_items.push_back(it.second);
    }
  }
  for (int q = 0; q < nranks; ++q) {
    if (q == rank) continue;
    std::vector<std::vector<std::pair<long long, int>>> theirs;
    items_for(q, theirs);
    s->send_counts[q] = (long long)theirs[rank].size();
  }
  // send items in peer order (a second pass keeps the peers' groups contiguous and ordered by rank)
  for (int q = 0; q < nranks; ++q) {
    if (q == rank) continue;
    std::vector<std::vector<std::pair<long long, int>>> theirs;
    items_for(q, theirs);
    for (auto &it : theirs[rank]) {
      s->send_items.push_back((int32_t)(it.first - s->begin));
      s->send_items.push_back(it.second);
    }
  }
  *out = s;
  return FX_OK;
}

extern "C" int fx_shard_destroy(fx_shard *s) {
  delete s;
  return FX_OK;
}

extern "C" int fx_shard_sizes(const fx_shard *s, int64_t *owned_begin, int64_t *n_owned, int64_t *n_ghost, int64_t *n_send,
                              int64_t *n_recv) {
  if (!s) return fx_fail(FX_ERR_INVALID_ARG, "shard_sizes: null shard");
  if (owned_begin) *owned_begin = s->begin;
  if (n_owned) *n_owned = s->end - s->begin;
  if (n_ghost) *n_ghost = (int64_t)s->ghosts.size();
  if (n_send) *n_send = (int64_t)s->send_items.size() / 2;
  if (n_recv) *n_recv = (int64_t)s->recv_items.size() / 2;
  return FX_OK;
}

extern "C" int fx_shard_tables(const fx_shard *s, int32_t *neigh_local, int64_t *global_id) {
  if (!s || !neigh_local || !global_id) return fx_fail(FX_ERR_INVALID_ARG, "shard_tables: null argument");
  std::copy(s->neigh_local.begin(), s->neigh_local.end(), neigh_local);
  const long long nown = s->end - s->begin;
  for (long long b = 0; b < nown; ++b) global_id[b] = s->begin + b;
  for (size_t g = 0; g < s->ghosts.size(); ++g) global_id[nown + (long long)g] = s->ghosts[g];
  return FX_OK;
}

extern "C" int fx_shard_items(const fx_shard *s, int32_t *send_items, int64_t *send_counts, int32_t *recv_items, int64_t *recv_counts) {
  if (!s || !send_counts || !recv_counts) return fx_fail(FX_ERR_INVALID_ARG, "shard_items: null argument");
  if (send_items) std::copy(s->send_items.begin(), s->send_items.end(), send_items);
  if (recv_items) std::copy(s->recv_items.begin(), s->recv_items.end(), recv_items);
  for (int p = 0; p < s->nranks; ++p) {
    send_counts[p] = s->send_counts[p];
    recv_counts[p] = s->recv_counts[p];
  }
  return FX_OK;
}

// ------------------------------------------------------------------ device: face slabs <-> packed buffer
// Item = (block, side): the R-deep slab of the block's INTERIOR next to face `side` (0 -x, 1 +x, 2 -y, 3 +y, 4 -z, 5 +z),
// all variables, laid out [v][k][j][i] over the slab's own extents (i fastest).  One CTA per item.
__device__ __forceinline__ void fx_slab_geometry(const FxParams &P, int side, int R, int e[3], int o[3]) {
  const int d = side >> 1;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    e[a] = P.n[a];
    o[a] = P.gd[a];
  }
  e[d] = R;
  if (side & 1) o[d] += P.n[d] - R;
}

// The copy of one slab with its extents known at compile time (16-wide blocks, depth 2: the PLM slabs of the fused path) and
// two doubles per thread: the element -> (v, k, j, i) decode is shifts and masks instead of three integer divisions per
// element, which were most of the kernel's instructions (0.51 ms per step for 126 MB of slabs each way on rank 0 of 8).
template <bool PACK, int E0, int E1, int E2>
__device__ __forceinline__ void fx_slab_copy_fixed(const FxParams &P, double *U, int b, const int o[3], double *dst) {
  constexpr int H0 = E0 / 2, PER = H0 * E1 * E2;  // pairs per row, per variable
  const int total = PER * P.nvars;
  for (int t = threadIdx.x; t < total; t += blockDim.x) {
    const int v = t / PER, c = t - v * PER;
    const int k = c / (H0 * E1), r2 = c - k * (H0 * E1);
    const int j = r2 / H0, i = 2 * (r2 - j * H0);
    const long long a = (long long)v * P.S_v + (long long)b * P.S_b + (long long)(k + o[2]) * P.S_k + (long long)(j + o[1]) * P.S_j + (i + o[0]);
    double2 *p = reinterpret_cast<double2 *>(U + a), *q = reinterpret_cast<double2 *>(dst) + t;
    if (PACK) *q = *p; else *p = *q;
  }
}

template <bool PACK>
__global__ void __launch_bounds__(256) fx_k_halo_slabs(const FxParams P, double *U, const int *__restrict__ items,
                                                       const long long *__restrict__ offsets, int R, double *buf) {
  const long long it = blockIdx.x;
  const int b = items[2 * it], side = items[2 * it + 1];
  int e[3], o[3];
  fx_slab_geometry(P, side, R, e, o);
  double *dst = buf + offsets[it];
  // the fixed-extent form needs 16-byte aligned pairs: even origins and strides (even guard depths), an aligned array and slot
  const bool pairs = R == 2 && P.n[0] == 16 && P.n[1] == 16 && P.n[2] == 16 && !((o[0] | P.S_j) & 1) &&
                     !(((unsigned long long)U | (unsigned long long)dst) & 15);
  if (pairs) {
    const int d = side >> 1;
    if (d == 0) fx_slab_copy_fixed<PACK, 2, 16, 16>(P, U, b, o, dst);
    else if (d == 1) fx_slab_copy_fixed<PACK, 16, 2, 16>(P, U, b, o, dst);
    else fx_slab_copy_fixed<PACK, 16, 16, 2>(P, U, b, o, dst);
    return;
  }
  const int per_var = e[0] * e[1] * e[2];
  const int total = per_var * P.nvars;
  for (int t = threadIdx.x; t < total; t += blockDim.x) {
    const int v = t / per_var, c = t - v * per_var;
    const int k = c / (e[0] * e[1]), r2 = c - k * e[0] * e[1];
    const int j = r2 / e[0], i = r2 - j * e[0];
    const long long a = (long long)v * P.S_v + (long long)b * P.S_b + (long long)(k + o[2]) * P.S_k + (long long)(j + o[1]) * P.S_j + (i + o[0]);
    if (PACK) dst[t] = U[a]; else U[a] = dst[t];
  }
}

static int fx_halo_depth(const fx_hydro_plan *plan) { return plan->P.recon == FX_RECON_WENO5 ? 3 : 2; }

extern "C" int64_t fx_halo_item_elems(const fx_hydro_plan *plan, int side) {
  if (!plan || side < 0 || side > 5) return -1;
  const int d = side >> 1;
  if (!plan->P.active[d]) return 0;
  long long n = plan->nvars;
  for (int a = 0; a < 3; ++a) n *= (a == d) ? fx_halo_depth(plan) : plan->P.n[a];
  return n;
}

static int fx_halo_launch(fx_hydro_plan *plan, double *U, const int32_t *items, const int64_t *offsets, int64_t n, double *buf,
                          bool pack, void *stream) {
  if (!plan) return fx_fail(FX_ERR_INVALID_ARG, "halo pack/unpack: null plan");
  if (n < 0 || (n > 0 && (!U || !items || !offsets || !buf))) return fx_fail(FX_ERR_INVALID_ARG, "halo pack/unpack: null argument");
  if (n == 0) return FX_OK;
  if (n > 0x7fffffffLL) return fx_fail(FX_ERR_INVALID_ARG, "halo pack/unpack: too many items");
  const int R = fx_halo_depth(plan);
  if (pack) fx_k_halo_slabs<true><<<(unsigned)n, 256, 0, (cudaStream_t)stream>>>(plan->P, U, items, (const long long *)offsets, R, buf);
  else fx_k_halo_slabs<false><<<(unsigned)n, 256, 0, (cudaStream_t)stream>>>(plan->P, U, items, (const long long *)offsets, R, buf);
  FX_LAUNCH_CHECK("halo_slabs");
  return FX_OK;
}

extern "C" int fx_halo_pack(fx_hydro_plan *plan, const double *U, const int32_t *items_dev, const int64_t *offsets_dev, int64_t n,
                            double *buf, void *stream) {
  return fx_halo_launch(plan, const_cast<double *>(U), items_dev, offsets_dev, n, buf, true, stream);
}

extern "C" int fx_halo_unpack(fx_hydro_plan *plan, double *U, const int32_t *items_dev, const int64_t *offsets_dev, int64_t n,
                              const double *buf, void *stream) {
  return fx_halo_launch(plan, U, items_dev, offsets_dev, n, const_cast<double *>(buf), false, stream);
}
