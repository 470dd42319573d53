// tfa_shard.cu — SURVEY 8(f)4 / 8(e): sharding of the assembly over several GPUs (the way past one device's
// memory the paper names, L26: the Jacobian of config 5 is 41 GB).
//
// Rows are independent given neighbour data, so each rank owns a contiguous chunk of the (RCM-ordered) cells, its
// rows of the BSR matrix and of rhs, and keeps read-only copies ("ghosts") of the cells its stencils reach.  One
// assembly needs two neighbour-only exchanges and no reduction:
//   (1) before the gradient kernel: the states of the ghost cells (the vertex-neighbour layer of the owned cells);
//   (2) between the two kernels: the reconstructed face states (F x 18 doubles) of the ghost cells that are FACE
//       neighbours of owned cells.  Those ghost cells are run through the face lanes of k_assemble as well: cell i
//       evaluates the block (j,i) of its neighbour's row, so an owned row j gets its ghost-column
//       blocks from the ghost cell's lanes; the ghost's own diagonal block and its blocks towards cells of other
//       ranks have no target here (block map -1) and its faces towards them are closed (transmissive on its own,
//       valid, face state), so nothing undefined is ever read.
// The local cells keep the ORDER of their global ids (ghosts below the owned range, the owned range, ghosts above):
// stencil order, BSR column order, a face's L/R choice and its numbering by node pair are then those of the global
// mesh, and an owned row comes out bit-identical to the single-GPU assembly.
//
// tfa_partition_* is host-only logic on host arrays (testable without a GPU); tfa_shard_* builds the local mesh
// and the device tables from a global tfa_mesh; the exchanges themselves are the caller's (NCCL send/recv through
// torch.distributed in api.py), between this library's pack / unpack kernels.
#include <algorithm>
#include <new>
#include <vector>

#include "tfa_common.cuh"

namespace tfa {
int build_mesh(tfa_mesh& m, cudaStream_t st);
int refresh_nbrf(tfa_mesh& m, cudaStream_t st);
}  // namespace tfa

struct tfa_partition {
  int n_ranks = 1, rank = 0;
  int64_t nc_global = 0, c0 = 0, c1 = 0;    // owned global range [c0, c1)
  std::vector<int32_t> l2g;                 // local -> global, ascending
  int64_t o0 = 0;                           // local id of the first owned cell (owned = [o0, o0 + c1 - c0))
  // per peer, ascending global id on both sides (the relations are symmetric, so sender and receiver agree)
  std::vector<std::vector<int32_t>> send_state, recv_state;   // local ids: owned cells a peer's stencils reach /
                                                              // ghosts owned by that peer
  std::vector<std::vector<int32_t>> send_face, recv_face;     // the same for face neighbours only
  int64_t n_local() const { return (int64_t)l2g.size(); }
  int64_t n_owned() const { return c1 - c0; }
};

namespace {
inline int64_t chunk_begin(int64_t nc, int n, int r) { return nc * (int64_t)r / n; }
inline int owner_of(int64_t nc, int n, int64_t g) {
  int r = (int)((g * n + n - 1) / nc);     // first guess, then adjust to chunk_begin(r) <= g < chunk_begin(r+1)
  if (r >= n) r = n - 1;
  while (r > 0 && g < chunk_begin(nc, n, r)) --r;
  while (r + 1 < n && g >= chunk_begin(nc, n, r + 1)) ++r;
  return r;
}
}  // namespace

extern "C" {

int tfa_partition_create(tfa_partition** out, int64_t n_cells, int max_faces, const int32_t* cell_nbr,
                         const int32_t* stencil_ptr, const int32_t* stencil_idx, int n_ranks, int rank) {
  using tfa::set_error;
  if (!out || n_cells < 0 || (max_faces != 3 && max_faces != 4) || n_ranks < 1 || rank < 0 || rank >= n_ranks ||
      (n_cells > 0 && (!cell_nbr || !stencil_ptr || !stencil_idx)))
    return set_error(TFA_EINVAL, "tfa_partition_create: bad argument");
  tfa_partition* p = new (std::nothrow) tfa_partition;
  if (!p) return set_error(TFA_ENOMEM, "host allocation failed");
  const int F = max_faces;
  p->n_ranks = n_ranks;
  p->rank = rank;
  p->nc_global = n_cells;
  p->c0 = chunk_begin(n_cells, n_ranks, rank);
  p->c1 = chunk_begin(n_cells, n_ranks, rank + 1);
  const int64_t c0 = p->c0, c1 = p->c1;
  // ghosts = vertex neighbours of owned cells that are not owned (L74: the reconstruction stencil)
  std::vector<int32_t> ghosts;
  for (int64_t i = c0; i < c1; ++i)
    for (int32_t q = stencil_ptr[i]; q < stencil_ptr[i + 1]; ++q) {
      const int32_t j = stencil_idx[q];
      if (j < c0 || j >= c1) ghosts.push_back(j);
    }
  std::sort(ghosts.begin(), ghosts.end());
  ghosts.erase(std::unique(ghosts.begin(), ghosts.end()), ghosts.end());
  const auto mid = std::lower_bound(ghosts.begin(), ghosts.end(), (int32_t)c0);
  p->o0 = mid - ghosts.begin();
  p->l2g.assign(ghosts.begin(), mid);
  for (int64_t i = c0; i < c1; ++i) p->l2g.push_back((int32_t)i);
  p->l2g.insert(p->l2g.end(), mid, ghosts.end());
  auto local_of = [&](int32_t g) -> int32_t {
    if (g >= c0 && g < c1) return (int32_t)(p->o0 + (g - c0));
    return (int32_t)(std::lower_bound(p->l2g.begin(), p->l2g.end(), g) - p->l2g.begin());
  };
  p->send_state.assign(n_ranks, {});
  p->recv_state.assign(n_ranks, {});
  p->send_face.assign(n_ranks, {});
  p->recv_face.assign(n_ranks, {});
  // receive lists: my ghosts by owner (ascending global id = ascending local id)
  std::vector<char> face_ghost(ghosts.size(), 0);
  for (int64_t i = c0; i < c1; ++i)
    for (int k = 0; k < F; ++k) {
      const int32_t j = cell_nbr[F * i + k];
      if (j >= 0 && (j < c0 || j >= c1))
        face_ghost[std::lower_bound(ghosts.begin(), ghosts.end(), j) - ghosts.begin()] = 1;
    }
  for (size_t q = 0; q < ghosts.size(); ++q) {
    const int r = owner_of(n_cells, n_ranks, ghosts[q]);
    p->recv_state[r].push_back(local_of(ghosts[q]));
    if (face_ghost[q]) p->recv_face[r].push_back(local_of(ghosts[q]));
  }
  // send lists: an owned cell goes to every rank that owns one of its vertex (face) neighbours
  std::vector<int> seen(n_ranks, -1);
  for (int64_t i = c0; i < c1; ++i) {
    for (int32_t q = stencil_ptr[i]; q < stencil_ptr[i + 1]; ++q) {
      const int32_t j = stencil_idx[q];
      if (j >= c0 && j < c1) continue;
      const int r = owner_of(n_cells, n_ranks, j);
      if (seen[r] != (int)(i - c0)) { seen[r] = (int)(i - c0); p->send_state[r].push_back(local_of((int32_t)i)); }
    }
  }
  std::fill(seen.begin(), seen.end(), -1);
  for (int64_t i = c0; i < c1; ++i)
    for (int k = 0; k < F; ++k) {
      const int32_t j = cell_nbr[F * i + k];
      if (j < 0 || (j >= c0 && j < c1)) continue;
      const int r = owner_of(n_cells, n_ranks, j);
      if (seen[r] != (int)(i - c0)) { seen[r] = (int)(i - c0); p->send_face[r].push_back(local_of((int32_t)i)); }
    }
  *out = p;
  return 0;
}

void tfa_partition_destroy(tfa_partition* p) { delete p; }

int tfa_partition_sizes(const tfa_partition* p, int64_t* n_local, int64_t* n_owned, int64_t* first_owned_local,
                        int64_t* first_owned_global) {
  if (!p) return tfa::set_error(TFA_EINVAL, "null partition");
  if (n_local) *n_local = p->n_local();
  if (n_owned) *n_owned = p->n_owned();
  if (first_owned_local) *first_owned_local = p->o0;
  if (first_owned_global) *first_owned_global = p->c0;
  return 0;
}

static const std::vector<int32_t>* part_list(const tfa_partition* p, int which, int peer) {
  if (which == TFA_PART_LOCAL_TO_GLOBAL) return &p->l2g;
  if (peer < 0 || peer >= p->n_ranks) return nullptr;
  switch (which) {
    case TFA_PART_SEND_STATE: return &p->send_state[peer];
    case TFA_PART_RECV_STATE: return &p->recv_state[peer];
    case TFA_PART_SEND_FACE: return &p->send_face[peer];
    case TFA_PART_RECV_FACE: return &p->recv_face[peer];
    default: return nullptr;
  }
}

int64_t tfa_partition_count(const tfa_partition* p, int which, int peer) {
  if (!p) return -1;
  const std::vector<int32_t>* v = part_list(p, which, peer);
  return v ? (int64_t)v->size() : -1;
}

int tfa_partition_get(const tfa_partition* p, int which, int peer, int32_t* host_dst, int64_t count) {
  if (!p || (!host_dst && count > 0)) return tfa::set_error(TFA_EINVAL, "null argument");
  const std::vector<int32_t>* v = part_list(p, which, peer);
  if (!v) return tfa::set_error(TFA_EINVAL, "tfa_partition_get: unknown list or peer");
  if ((int64_t)v->size() != count) return tfa::set_error(TFA_EINVAL, "tfa_partition_get: count mismatch");
  std::copy(v->begin(), v->end(), host_dst);
  return 0;
}

}  // extern "C"

// ================================================================================================
// device side: the local mesh of a rank, its tables, pack / unpack of the two halos
// ================================================================================================
struct tfa_shard {
  tfa_partition* part = nullptr;
  tfa_mesh* mesh = nullptr;                 // owned + ghost cells, local ids ascending in global id
  int64_t nnzb_owned = 0, block_offset = 0; // the owned rows' blocks are [block_offset, block_offset + nnzb_owned)
                                            // of the local pattern; the shard's value array starts at block_offset
  std::vector<int32_t> bface_global;        // [nb_local] global boundary-face index, -1 on a cut face
  std::vector<tfa::DevBuf<int32_t>> d_send[2], d_recv[2];   // [kind][peer] device copies of the lists
  ~tfa_shard() {
    delete part;
    delete mesh;
  }
};

namespace tfa {
int create_mesh_from_padded(tfa_mesh** out, int64_t n_nodes, const double* node_xy, int64_t n_cells, int F,
                            const int32_t* cell_nodes, const double* cell_xy, cudaStream_t st);

namespace {
constexpr int TPB = 256;

// Tables of a rank's local mesh: a ghost cell closes every face that does not lead to an owned cell (transmissive
// on its own face state) and keeps only the blocks it writes into owned rows; block indices become relative to the
// first owned row's first block.
__global__ void k_shard_tables(int64_t nl, int F, int BS, int64_t o0, int64_t o1, int32_t off,
                               const int32_t* __restrict__ cell_nbr, int32_t* __restrict__ nbrf,
                               int32_t* __restrict__ blkmap, int32_t* __restrict__ pblkmap) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nl) return;
  const bool own = i >= o0 && i < o1;
  int32_t* b = blkmap + BS * i;
  int32_t* pb = pblkmap + BS * i;
  b[0] = own ? b[0] - off : -1;
  // packed form of the owned rows: diagonal blocks indexed by the owned cell, off-diagonal blocks in the order of
  // the owned rows' pattern with the diagonal ones taken out (columns ascend in local id, so the mirror block
  // (j, i) lies behind row j's diagonal block exactly when i > j)
  pb[0] = own ? (int32_t)(i - o0) : -1;
  for (int k = 0; k < F; ++k) {
    const int64_t j = cell_nbr[F * i + k];
    const bool to_owned = j >= o0 && j < o1;
    b[1 + k] = (to_owned && b[1 + k] >= 0) ? b[1 + k] - off : -1;
    pb[1 + k] = b[1 + k] >= 0 ? b[1 + k] - (int32_t)(j - o0) - (i > j ? 1 : 0) : -1;
    if (!own && !to_owned) nbrf[F * i + k] = -1;
  }
}

__global__ void k_pack_rows(int64_t n, int w2, const int32_t* __restrict__ idx, const double2* __restrict__ src,
                            double2* __restrict__ buf) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= n * w2) return;
  const int64_t r = t / w2;
  const int c = (int)(t - r * w2);
  buf[t] = src[(int64_t)idx[r] * w2 + c];
}
__global__ void k_unpack_rows(int64_t n, int w2, const int32_t* __restrict__ idx, const double2* __restrict__ buf,
                              double2* __restrict__ dst) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= n * w2) return;
  const int64_t r = t / w2;
  const int c = (int)(t - r * w2);
  dst[(int64_t)idx[r] * w2 + c] = buf[t];
}

template <class T>
int download(const DevBuf<T>& d, int64_t n, std::vector<T>& h, cudaStream_t st) {
  h.resize((size_t)std::max<int64_t>(n, 0));
  if (n > 0) TFA_CUDA(cudaMemcpyAsync(h.data(), d.p, (size_t)n * sizeof(T), cudaMemcpyDeviceToHost, st));
  return 0;
}
}  // namespace
}  // namespace tfa

using namespace tfa;

extern "C" {

int tfa_shard_create(tfa_shard** out, const tfa_mesh* g, int n_ranks, int rank, void* stream) {
  if (!out || !g || n_ranks < 1 || rank < 0 || rank >= n_ranks) return set_error(TFA_EINVAL, "tfa_shard_create: bad argument");
  cudaStream_t st = (cudaStream_t)stream;
  const int F = g->F, BS = blk_stride(F);
  const int64_t nc = g->nc;
  std::vector<int32_t> nbr, sp, si, cn, fnodes, bfof, tags;
  std::vector<double> cx, nxy;
  TFA_TRY(download(g->cell_nbr, F * nc, nbr, st));
  TFA_TRY(download(g->st_ptr, nc + 1, sp, st));
  TFA_TRY(download(g->st_idx, g->nst, si, st));
  TFA_TRY(download(g->cell_nodes, F * nc, cn, st));
  TFA_TRY(download(g->cell_xy, 2 * F * nc, cx, st));
  TFA_TRY(download(g->node_xy, 2 * g->nn, nxy, st));
  TFA_TRY(download(g->face_nodes, 2 * g->nf, fnodes, st));
  TFA_TRY(download(g->bface_of, g->nf, bfof, st));
  TFA_TRY(download(g->bc_tag, g->nb, tags, st));
  TFA_CUDA(cudaStreamSynchronize(st));
  tfa_shard* s = new (std::nothrow) tfa_shard;
  if (!s) return set_error(TFA_ENOMEM, "host allocation failed");
  auto body = [&]() -> int {
    TFA_TRY(tfa_partition_create(&s->part, nc, F, nbr.data(), sp.data(), si.data(), n_ranks, rank));
    const tfa_partition& P = *s->part;
    const int64_t nl = P.n_local();
    std::vector<int32_t> lcn((size_t)F * nl);
    std::vector<double> lcx((size_t)2 * F * nl);
    for (int64_t l = 0; l < nl; ++l) {
      const int64_t gi = P.l2g[l];
      std::copy(cn.begin() + F * gi, cn.begin() + F * (gi + 1), lcn.begin() + F * l);
      std::copy(cx.begin() + 2 * F * gi, cx.begin() + 2 * F * (gi + 1), lcx.begin() + 2 * F * l);
    }
    TFA_TRY(create_mesh_from_padded(&s->mesh, g->nn, nxy.data(), nl, F, lcn.data(), lcx.data(), st));
    tfa_mesh& m = *s->mesh;
    // boundary rules: a local boundary face is a boundary face of the global mesh (same node pair: it keeps its
    // tag and its place in the caller's ghost-state array) or a cut (closed; never evaluated for an owned cell)
    std::vector<int32_t> lbf, lfn;
    TFA_TRY(download(m.bfaces, m.nb, lbf, st));
    TFA_TRY(download(m.face_nodes, 2 * m.nf, lfn, st));
    TFA_CUDA(cudaStreamSynchronize(st));
    s->bface_global.assign((size_t)m.nb, -1);
    std::vector<int32_t> ltags((size_t)m.nb, TFA_BC_TRANSMISSIVE);
    const int64_t nn = g->nn;
    auto key = [&](const int32_t* e) { return (int64_t)e[0] * nn + e[1]; };
    for (int64_t b = 0; b < m.nb; ++b) {
      const int64_t want = key(&lfn[2 * (size_t)lbf[b]]);
      int64_t lo = 0, hi = g->nf;   // global faces are sorted by this key
      while (lo < hi) {
        const int64_t mid = (lo + hi) / 2;
        if (key(&fnodes[2 * mid]) < want) lo = mid + 1; else hi = mid;
      }
      if (lo >= g->nf || key(&fnodes[2 * lo]) != want) return set_error(TFA_EMESH, "shard face not found in the global mesh");
      const int32_t gb = bfof[lo];
      if (gb >= 0) { s->bface_global[b] = gb; ltags[b] = tags[gb]; }
    }
    TFA_TRY(tfa_mesh_set_bc(&m, ltags.data(), stream));
    m.shard_local = true;
    // block offset of the owned rows, then the shard's tables
    std::vector<int32_t> rp;
    TFA_TRY(download(m.bsr_rowptr, nl + 1, rp, st));
    TFA_CUDA(cudaStreamSynchronize(st));
    const int64_t o0 = P.o0, o1 = P.o0 + P.n_owned();
    s->block_offset = nl ? rp[o0] : 0;
    s->nnzb_owned = nl ? rp[o1] - rp[o0] : 0;
    if (nl) {
      k_shard_tables<<<cdiv(nl, TPB), TPB, 0, st>>>(nl, F, BS, o0, o1, (int32_t)s->block_offset, m.cell_nbr.p, m.nbrf.p,
                                                   m.blkmap.p, m.pblkmap.p);
      TFA_CUDA(cudaGetLastError());
    }
    for (int kind = 0; kind < 2; ++kind) {
      s->d_send[kind] = std::vector<DevBuf<int32_t>>(n_ranks);
      s->d_recv[kind] = std::vector<DevBuf<int32_t>>(n_ranks);
      for (int r = 0; r < n_ranks; ++r) {
        const std::vector<int32_t>& a = kind == 0 ? P.send_state[r] : P.send_face[r];
        const std::vector<int32_t>& b = kind == 0 ? P.recv_state[r] : P.recv_face[r];
        TFA_CUDA(s->d_send[kind][r].alloc((int64_t)a.size()));
        TFA_CUDA(s->d_recv[kind][r].alloc((int64_t)b.size()));
        if (!a.empty()) TFA_CUDA(cudaMemcpyAsync(s->d_send[kind][r].p, a.data(), a.size() * 4, cudaMemcpyHostToDevice, st));
        if (!b.empty()) TFA_CUDA(cudaMemcpyAsync(s->d_recv[kind][r].p, b.data(), b.size() * 4, cudaMemcpyHostToDevice, st));
      }
    }
    TFA_CUDA(cudaStreamSynchronize(st));
    return 0;
  };
  const int rc = body();
  if (rc) { delete s; return rc; }
  *out = s;
  return 0;
}

void tfa_shard_destroy(tfa_shard* s) { delete s; }
const tfa_mesh* tfa_shard_mesh(const tfa_shard* s) { return s ? s->mesh : nullptr; }
const tfa_partition* tfa_shard_partition(const tfa_shard* s) { return s ? s->part : nullptr; }

int tfa_shard_info(const tfa_shard* s, int64_t* nnzb_owned, int64_t* block_offset) {
  if (!s) return set_error(TFA_EINVAL, "null shard");
  if (nnzb_owned) *nnzb_owned = s->nnzb_owned;
  if (block_offset) *block_offset = s->block_offset;
  return 0;
}

int tfa_shard_bface_global(const tfa_shard* s, int32_t* host_dst, int64_t count) {
  if (!s || (!host_dst && count > 0)) return set_error(TFA_EINVAL, "null argument");
  if (count != (int64_t)s->bface_global.size()) return set_error(TFA_EINVAL, "tfa_shard_bface_global: count mismatch");
  std::copy(s->bface_global.begin(), s->bface_global.end(), host_dst);
  return 0;
}

// the list of one halo exchange, or NULL for a bad shard / kind / peer
static const std::vector<int32_t>* halo_list(const tfa_shard* s, int kind, int peer, bool send) {
  if (!s || (kind != TFA_HALO_STATE && kind != TFA_HALO_FACE) || peer < 0 || peer >= s->part->n_ranks) return nullptr;
  const tfa_partition& P = *s->part;
  if (kind == TFA_HALO_STATE) return send ? &P.send_state[peer] : &P.recv_state[peer];
  return send ? &P.send_face[peer] : &P.recv_face[peer];
}

// buf[r] = row send_list[r] of src; rows are 18 doubles (TFA_HALO_STATE) or F x 18 doubles (TFA_HALO_FACE)
int tfa_shard_pack(const tfa_shard* s, int kind, int peer, const double* src, double* buf, void* stream) {
  const std::vector<int32_t>* lst = halo_list(s, kind, peer, true);
  if (!lst) return set_error(TFA_EINVAL, "tfa_shard_pack: bad shard, kind or peer");
  if (lst->empty()) return 0;
  if (!src || !buf) return set_error(TFA_EINVAL, "tfa_shard_pack: null buffer");
  const int w2 = (kind == TFA_HALO_STATE ? NEQ : s->mesh->F * NEQ) / 2;
  const int64_t cnt = (int64_t)lst->size();
  k_pack_rows<<<cdiv(cnt * w2, TPB), TPB, 0, (cudaStream_t)stream>>>(cnt, w2, s->d_send[kind][peer].p,
                                                                    (const double2*)src, (double2*)buf);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

// row recv_list[r] of dst = buf[r]
int tfa_shard_unpack(const tfa_shard* s, int kind, int peer, const double* buf, double* dst, void* stream) {
  const std::vector<int32_t>* lst = halo_list(s, kind, peer, false);
  if (!lst) return set_error(TFA_EINVAL, "tfa_shard_unpack: bad shard, kind or peer");
  if (lst->empty()) return 0;
  if (!buf || !dst) return set_error(TFA_EINVAL, "tfa_shard_unpack: null buffer");
  const int w2 = (kind == TFA_HALO_STATE ? NEQ : s->mesh->F * NEQ) / 2;
  const int64_t cnt = (int64_t)lst->size();
  k_unpack_rows<<<cdiv(cnt * w2, TPB), TPB, 0, (cudaStream_t)stream>>>(cnt, w2, s->d_recv[kind][peer].p,
                                                                      (const double2*)buf, (double2*)dst);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

}  // extern "C"
