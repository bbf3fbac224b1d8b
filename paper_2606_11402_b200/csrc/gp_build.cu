// Plain GPU graph builder.  Separately timed.
//
//   b1 order   bit-reversed left-balanced k-d tree: node i at level l = floor(log2(i+1)),
//              position p = i - (2^l - 1), children i + 2^l (left) and i + 2^(l+1) (right).  Built level
//              by level: one global radix sort per level by (subtree id, rank of the point along
//              dimension l mod d); the element at offset S(left child) of its subtree becomes the node.
//              Ranks are dense (coordinate, user id) ranks, so ties are broken by user id (R-4).
//   b2 kNN     per query i: depth-first walk of the tree restricted to nodes < i (every prefix of the
//              order is itself a valid tree), candidates ranked by (fp64 FMA-free squared
//              distance, tree index) (R-5).  One thread per query, queries of one warp are
//              spatial neighbours (heap-order enumeration of each level).
//   b3 depth   d_i = 1 + max_{j in c(i)} d_j: the fixed point of PAPER.md:59, reached in one dataflow launch.
//   b4 sort    stable sort of tree indices by depth (optionally by Morton code inside a depth), remap.
//
// Sorting and scanning use CUB (a library primitive on a path that is not the hot path).
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_partition.cuh>

#include "gp_common.cuh"

namespace gp {

struct BuildLayout {
  size_t ctrl, rank, keys_a, keys_b, vals_a, vals_b, seg, perm_tree, x_tree, nbr_tree, depth_tree, tree2pos,
      pos2tree, bbox, boff, cub_tmp, cub_bytes, total;
};

static BuildLayout build_layout(int64_t n, int d, int k, int dtype) {
  BuildLayout L{};
  size_t B = dtype_bytes(dtype), N = (size_t)n, off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes, 256); return o; };
  L.ctrl = take(kCtrlBytes);
  L.rank = take(N * 4 * d);
  L.keys_a = take(N * 8);
  L.keys_b = take(N * 8);
  L.vals_a = take(N * 4);
  L.vals_b = take(N * 4);
  L.seg = take(N * 4);
  L.perm_tree = take(N * 4);
  L.x_tree = take(N * d * B);
  L.nbr_tree = take(N * (size_t)k * 4);
  L.depth_tree = take(N * 4);
  L.tree2pos = take(N * 4);
  L.pos2tree = take(N * 4);
  L.bbox = take(256);
  L.boff = take(((size_t)kMaxBatches + 2) * 8);
  L.cub_bytes = (64u << 20) + N / 2;
  L.cub_tmp = take(L.cub_bytes);
  L.total = off;
  return L;
}

// ---- small helpers ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t order_bits(float f) {
  f += 0.0f;  // -0 -> +0
  uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ uint64_t order_bits(double f) {
  f += 0.0;
  uint64_t u = (uint64_t)__double_as_longlong(f);
  return (u & 0x8000000000000000ULL) ? ~u : (u | 0x8000000000000000ULL);
}

template <typename T, typename KeyT>
__global__ void coord_keys_kernel(const T* __restrict__ x, int64_t n, int d, int dim, KeyT* __restrict__ keys,
                                  uint32_t* __restrict__ ids) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  keys[i] = (KeyT)order_bits(x[i * d + dim]);
  ids[i] = (uint32_t)i;
}

__global__ void scatter_rank_kernel(const uint32_t* __restrict__ sorted_ids, int64_t n, uint32_t* __restrict__ rank) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n) rank[sorted_ids[p]] = (uint32_t)p;
}

__global__ void iota_seg_kernel(uint32_t* __restrict__ ids, uint32_t* __restrict__ seg, int64_t n) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { ids[i] = (uint32_t)i; seg[i] = 0u; }
}

__global__ void level_keys_kernel(const uint32_t* __restrict__ ids, const uint32_t* __restrict__ seg,
                                  const uint32_t* __restrict__ rank_dim, int64_t m, int rank_bits,
                                  uint64_t* __restrict__ keys) {
  int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e < m) keys[e] = ((uint64_t)seg[e] << rank_bits) | (uint64_t)rank_dim[ids[e]];
}

// Tree shape of an N-node prefix (R-2): levels 0..Lam-1 full, level Lam holds positions 0..mlast-1.
struct TreeShape {
  int64_t n;
  int lam;        // level of node n-1
  int64_t mlast;  // nodes on the last level
};
__host__ __device__ inline TreeShape tree_shape(int64_t n) {
  TreeShape s; s.n = n; int l = 0;
  while (((int64_t)1 << (l + 1)) - 1 < n) ++l;   // smallest l with 2^(l+1) - 1 >= n
  s.lam = l; s.mlast = n - (((int64_t)1 << l) - 1);
  return s;
}
// nodes of the last level lying in the subtree rooted at (l, p): positions q < mlast with q mod 2^l == p
__host__ __device__ inline int64_t last_level_in(const TreeShape& s, int l, int64_t p) {
  int64_t step = (int64_t)1 << l;
  return p < s.mlast ? (s.mlast - p + step - 1) >> l : 0;       // step is a power of two: shifts, not divisions
}
__host__ __device__ inline int64_t subtree_size(const TreeShape& s, int l, int64_t p) {
  if (l > s.lam) return 0;
  if (l == s.lam) return p < s.mlast ? 1 : 0;
  return (((int64_t)1 << (s.lam - l)) - 1) + last_level_in(s, l, p);
}
// elements in subtrees (l, 0..p-1)
__host__ __device__ inline int64_t subtree_prefix(const TreeShape& s, int l, int64_t p) {
  int64_t step = (int64_t)1 << l;
  int64_t rem = s.mlast & (step - 1);
  int64_t last = (s.mlast >> l) * p + (rem < p ? rem : p);
  if (l == s.lam) return last;
  return p * (((int64_t)1 << (s.lam - l)) - 1) + last;
}

// After the level-l sort: element e of subtree (l, p) at offset q inside it goes left (q < S_left), becomes
// node (l, p) (q == S_left) or goes right.
__global__ void level_split_kernel(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ ids,
                                   int64_t m, int rank_bits, int l, TreeShape shape, uint32_t* __restrict__ seg_out,
                                   uint32_t* __restrict__ perm_tree) {
  int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= m) return;
  int64_t p = (int64_t)(keys[e] >> rank_bits);
  int64_t q = e - subtree_prefix(shape, l, p);
  int64_t sl = subtree_size(shape, l + 1, p);
  uint32_t out;
  if (q < sl) out = (uint32_t)p;
  else if (q == sl) { perm_tree[(((int64_t)1 << l) - 1) + p] = ids[e]; out = (uint32_t)((int64_t)2 << l); }  // retired
  else out = (uint32_t)(p + ((int64_t)1 << l));
  seg_out[e] = out;
}

// ---- b1, fast form: presorted lists, one stable partition per level -------------------------------------------------
// The plain order stage above re-sorts all active points by (subtree, coordinate rank) at every level: ceil(log2 N)
// radix sorts of 64-bit keys.  Sorting is needed only ONCE per dimension (the sort-based k-d build the paper points
// to): keep, for every dimension a, the list of active point ids grouped by subtree and sorted by
// (coordinate a, user id) inside each subtree.  At level l the list of the split dimension l mod d names every
// subtree's median by POSITION (offset = size of its left subtree, known in closed form for the left-balanced tree in
// bit-reversed numbering, R-2 / PAPER.md:39-41), which gives every point its side; then each list is split
// stably.  In the bit-reversed numbering the left child of subtree (l, p) is (l + 1, p) and the right child
// (l + 1, p + 2^l), so the level-(l + 1) list is [all left parts, in subtree order][all right parts, in
// subtree order]: the per-subtree split IS one global stable three-way partition (left / right / retired median) of the
// whole list, a single-pass cub::DevicePartition::If.  Order and ties are those of the plain stage (ranks ARE positions
// in these lists), hence of the oracle, bit for bit.
__host__ __device__ inline int64_t segment_of(const TreeShape& s, int l, int64_t e, int64_t* q) {
  // position e of a level-l list -> subtree p (bit-reversed position) and offset q inside it: the first r subtrees
  // hold base + 1 points, the others base (subtree_prefix inverted)
  const int64_t step = (int64_t)1 << l;
  const int64_t full = l < s.lam ? (((int64_t)1 << (s.lam - l)) - 1) : 0;
  const int64_t base = full + (s.mlast >> l), r = s.mlast & (step - 1);
  // everything is below 2^31 (n < 2^31): 32-bit divisions
  if (e < r * (base + 1)) { const uint32_t p = (uint32_t)e / (uint32_t)(base + 1); *q = e - (int64_t)p * (base + 1); return p; }
  const int64_t e2 = e - r * (base + 1);
  const uint32_t p2 = (uint32_t)e2 / (uint32_t)base;
  *q = e2 - (int64_t)p2 * base;
  return r + p2;
}

// Sides are kept as 2 bits per point id (0 left, 1 right, 2 = the point is node (l, p) and retires), 16 ids per word:
// every list looks the side of its ids up at random, and at N = 2^28 a byte per id (256 MB) no longer fits the L2
// while 64 MB does.  A thread owns the two bits of its id: it reads them plainly and flips what differs atomically.
__device__ __forceinline__ uint32_t side_get(const uint32_t* __restrict__ side, uint32_t id) {
  return (side[id >> 4] >> ((id & 15u) * 2u)) & 3u;
}

// split dimension's list: side of every active point
__global__ void level_classify_kernel(const uint32_t* __restrict__ lst, int64_t m, int l, TreeShape shape,
                                      uint32_t* __restrict__ side, uint32_t* __restrict__ perm_tree) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= m) return;
  int64_t q;
  const int64_t p = segment_of(shape, l, e, &q);
  const int64_t sl = subtree_size(shape, l + 1, p);
  const uint32_t id = lst[e];
  const uint32_t c = q < sl ? 0u : (q == sl ? 2u : 1u);
  const uint32_t old = side_get(side, id);
  if (old != c) atomicXor(&side[id >> 4], (old ^ c) << ((id & 15u) * 2u));
  if (c == 2u) perm_tree[(((int64_t)1 << l) - 1) + p] = id;
}

// selectors of the three-way stable partition (cub::DevicePartition::If): the id's side
struct SideIs {
  const uint32_t* side;
  uint32_t want;
  __device__ __forceinline__ bool operator()(const uint32_t& id) const { return side_get(side, id) == want; }
};

template <typename T>
__global__ void gather_points_kernel(const T* __restrict__ x_src, const uint32_t* __restrict__ idx, int64_t n, int d,
                                     T* __restrict__ x_dst) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int64_t s = idx[i];
  for (int t = 0; t < d; ++t) x_dst[i * d + t] = x_src[s * d + t];
}

__global__ void pack_points4_kernel(const float* __restrict__ x, int64_t n, int d, float4* __restrict__ x4) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
  v.x = x[i * d];
  if (d >= 2) v.y = x[i * d + 1];
  if (d >= 3) v.z = x[i * d + 2];
  x4[i] = v;
}

// ---- b2: preceding kNN --------------------------------------------------------------------------------
// canonical squared distance (R-5): double, left-to-right, no FMA contraction
template <typename T>
__device__ __forceinline__ double d2_canon(const double* xi, const T* __restrict__ xj, int d) {
  double acc = 0.0;
  for (int t = 0; t < d; ++t) {
    double dx = __dsub_rn(xi[t], (double)xj[t]);
    double sq = __dmul_rn(dx, dx);
    acc = t == 0 ? sq : __dadd_rn(acc, sq);
  }
  return acc;
}

template <typename T, int KMAX>
__global__ void __launch_bounds__(128)
knn_kernel(const T* __restrict__ x, int64_t n, int64_t n0, int d, int k, int64_t n_threads,
           int32_t* __restrict__ nbr, float* __restrict__ rad2, unsigned long long* __restrict__ overflow) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_threads) return;
  // thread t -> level l, heap position q -> bit-reversed position p -> tree index i: the queries of one
  // warp are consecutive leaves of the same level, i.e. spatial neighbours
  int l = 63 - __clzll((unsigned long long)(t + 1));
  int64_t q = t - (((int64_t)1 << l) - 1);
  int64_t p = l == 0 ? 0 : (int64_t)(__brevll((unsigned long long)q) >> (64 - l));
  int64_t i = (((int64_t)1 << l) - 1) + p;
  if (i >= n || i < n0) return;

  double xi[kMaxD];
  for (int a = 0; a < d; ++a) xi[a] = (double)x[i * d + a];
  double bd[KMAX];
  int32_t bi[KMAX];
  int cnt = 0, worst = 0;
  double wd = 0.0; int32_t wi = -1;

  // the walk pops one entry and pushes at most two children per node, so the stack never holds more than
  // (tree depth + 1) <= 32 entries for n < 2^31; a push that would not fit is COUNTED (the build then fails)
  struct Ent { int32_t node; double pd2; };
  constexpr int kStack = 40;
  Ent stack[kStack];
  int sp = 0;
  bool dropped = false;
  stack[sp++] = {0, 0.0};
  while (sp > 0) {
    Ent e = stack[--sp];
    if (cnt == k && e.pd2 > wd) continue;
    int32_t j = e.node;
    double dj = d2_canon<T>(xi, x + (int64_t)j * d, d);
    if (cnt < k) {
      bd[cnt] = dj; bi[cnt] = j; ++cnt;
      if (cnt == k) {
        worst = 0;
        for (int a = 1; a < k; ++a)
          if (bd[a] > bd[worst] || (bd[a] == bd[worst] && bi[a] > bi[worst])) worst = a;
        wd = bd[worst]; wi = bi[worst];
      }
    } else if (dj < wd || (dj == wd && j < wi)) {
      bd[worst] = dj; bi[worst] = j;
      worst = 0;
      for (int a = 1; a < k; ++a)
        if (bd[a] > bd[worst] || (bd[a] == bd[worst] && bi[a] > bi[worst])) worst = a;
      wd = bd[worst]; wi = bi[worst];
    }
    int lj = 31 - __clz(j + 1);
    int dim = lj % d;
    double diff = __dsub_rn(xi[dim], (double)x[(int64_t)j * d + dim]);
    int64_t left = (int64_t)j + ((int64_t)1 << lj), right = (int64_t)j + ((int64_t)2 << lj);
    int64_t near = diff < 0.0 ? left : right, far = diff < 0.0 ? right : left;
    double plane = __dmul_rn(diff, diff);
    if (far < i) { if (sp < kStack) stack[sp++] = {(int32_t)far, plane > e.pd2 ? plane : e.pd2}; else dropped = true; }
    if (near < i) { if (sp < kStack) stack[sp++] = {(int32_t)near, e.pd2}; else dropped = true; }
  }
  if (dropped) atomicAdd(overflow, 1ULL);
  // nearest first (selection sort on (d2, index))
  int32_t* out = nbr + (i - n0) * k;
  for (int a = 0; a < k; ++a) {
    int best = a;
    for (int b = a + 1; b < k; ++b)
      if (bd[b] < bd[best] || (bd[b] == bd[best] && bi[b] < bi[best])) best = b;
    double td = bd[a]; bd[a] = bd[best]; bd[best] = td;
    int32_t ti = bi[a]; bi[a] = bi[best]; bi[best] = ti;
    out[a] = bi[a];
  }
  rad2[i] = (float)bd[k - 1];   // squared neighbourhood radius: orders the points inside a batch (sort_keys_kernel)
}

// ---- b2, fast form: the same walk on shared memory ---------------------------------------------------------------
// Same walk as the plain kernel (pop, prune against the largest plane distance met on the way, visit, descend to the
// near child, park the far child), restructured after its profile (N = 2^24, config 3: 358 GB of DRAM traffic from the
// 830 bytes of local memory per thread): everything indexed at run time lives in SHARED memory, [slot][thread] so that
// a warp's accesses never conflict whatever slots its lanes are at - the stack (one fp32 bound, rounded DOWN, per
// level: see the kernel) and the k best (d^2, index) pairs as a max-heap whose root is the current
// k-th best, so accepting a candidate is one replace-root + sift-down (log2 k levels) instead of a rescan of all k.
// Result identical to the plain kernel, bit for bit (tests/test_gpu_builder.py).  Measured and dropped (DESIGN.md
// section 6.4): the stack-FREE traversal the paper points to (ref. Wald 2022b) with the list in registers,
// lanes that fetch their next query themselves, and a vote that reconverges the warp every visit.
// One warp per CTA: a CTA gives its shared memory back when its slowest warp is done, and the queries of different
// warps differ 2-3x in length on clustered inputs (measured at N = 2^24, kNN stage, CTAs of 128 / 64 / 32 threads:
// config 3 113 / 102 / 79 ms, config 4 81 / 66 / 64 ms).
constexpr int kKnnThreads = 32;

__device__ __forceinline__ bool key_gt(double da, int32_t ia, double db, int32_t ib) {
  return da > db || (da == db && ia > ib);
}

// max-heap of k (d^2, index) keys at hd[slot * kKnnThreads], hi[slot * kKnnThreads]: put (nd, ni) at the root and sift it down
__device__ __forceinline__ void heap_replace_root(double* hd, int32_t* hi, int k, double nd, int32_t ni) {
  int pos = 0;
  while (true) {
    const int c1 = 2 * pos + 1;
    if (c1 >= k) break;
    int c = c1;
    double dc = hd[c1 * kKnnThreads];
    int32_t ic = hi[c1 * kKnnThreads];
    if (c1 + 1 < k) {
      const double d2 = hd[(c1 + 1) * kKnnThreads];
      const int32_t i2 = hi[(c1 + 1) * kKnnThreads];
      if (key_gt(d2, i2, dc, ic)) { c = c1 + 1; dc = d2; ic = i2; }
    }
    if (!key_gt(dc, ic, nd, ni)) break;
    hd[pos * kKnnThreads] = dc;
    hi[pos * kKnnThreads] = ic;
    pos = c;
  }
  hd[pos * kKnnThreads] = nd;
  hi[pos * kKnnThreads] = ni;
}

// x4: for fp32 inputs the tree-ordered coordinates once more as one aligned 16-byte record per point ({x, y, z, 0}), so a
// node visit is one LDG.128 inside one sector instead of D scalar loads of a 4 D-byte record that straddles two sectors
// three times out of eight; nullptr for fp64 inputs.
template <typename T, int D, bool PACK4>
__global__ void __launch_bounds__(kKnnThreads)
knn_sm_kernel(const T* __restrict__ x, const float4* __restrict__ x4, int64_t n, int64_t n0, int k, int nlev,
              int64_t n_threads, int32_t* __restrict__ nbr, float* __restrict__ rad2) {
  extern __shared__ double knn_smem[];
  double* hd = knn_smem + threadIdx.x;                                                           // [k][kKnnThreads]
  int32_t* hi = reinterpret_cast<int32_t*>(knn_smem + (size_t)k * kKnnThreads) + threadIdx.x;     // [k][kKnnThreads]
  float* bnd = reinterpret_cast<float*>(hi - threadIdx.x + (size_t)k * kKnnThreads) + threadIdx.x;   // [nlev][kKnnThreads]
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_threads) return;
  // thread t -> level l, heap position q -> bit-reversed position p -> tree index i: the queries of one warp are
  // consecutive leaves of the same level, i.e. spatial neighbours
  const int l = 63 - __clzll((unsigned long long)(t + 1));
  const int64_t q = t - (((int64_t)1 << l) - 1);
  const int64_t p = l == 0 ? 0 : (int64_t)(__brevll((unsigned long long)q) >> (64 - l));
  const int64_t i = (((int64_t)1 << l) - 1) + p;
  if (i >= n || i < n0) return;

  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  double xi[D];
#pragma unroll
  for (int a = 0; a < D; ++a) xi[a] = (double)x[i * D + a];
  for (int a = 0; a < k; ++a) { hd[a * kKnnThreads] = inf; hi[a * kKnnThreads] = 0x7fffffff; }   // k sentinels: no separate fill phase
  double wd = inf;                             // root of the heap: the k-th best so far
  int32_t wi = 0x7fffffff;
  const uint32_t lim = (uint32_t)i;            // nodes < lim exist for this query (preceding points only)
  // The "stack": at most one parked sibling per level, and WHICH node it is follows from the path - node (level l,
  // position p) has children (l + 1, p) and (l + 1, p + 2^l), so bit t of p is the turn taken at level t and the
  // sibling parked at level L is (L, (p mod 2^(L-1)) + (1 - bit_{L-1}(p)) 2^(L-1)).  So only the BOUND of a parked
  // sibling is stored (fp32, [level][thread]) and a bit mask says which levels hold one: 4 bytes per level instead of
  // 8 per entry, which is what limits the warps per SM.  The deepest parked level is the top of the stack.
  uint32_t parked = 0;
  int32_t curr = 0;
  int lc = 0;                                  // level of curr
  float bound = 0.0f;                          // lower bound of d^2 for everything below curr
  bool have = true;
  while (true) {
    if (!have) {
      if (!parked) break;
      const int L = 31 - __clz(parked);
      parked &= ~(1u << L);
      const uint32_t p = (uint32_t)curr + 1u - (1u << lc), hb = 1u << (L - 1);
      curr = (int32_t)((2u * hb - 1u) + (p & (hb - 1u)) + ((p & hb) ^ hb));
      lc = L;
      bound = bnd[L * kKnnThreads];
      have = true;
    }
    if ((double)bound > wd) { have = false; continue; }
    double xn[D];
    if constexpr (PACK4) {
      const float4 v = __ldg(x4 + curr);
      xn[0] = (double)v.x;
      if (D >= 2) xn[1] = (double)v.y;
      if (D >= 3) xn[2] = (double)v.z;
    } else {
      const T* xc = x + (int64_t)curr * D;
#pragma unroll
      for (int a = 0; a < D; ++a) xn[a] = (double)__ldg(xc + a);
    }
    const int dim = lc % D;
    double acc = 0.0, diff = 0.0;
#pragma unroll
    for (int a = 0; a < D; ++a) {
      const double dx = __dsub_rn(xi[a], xn[a]);
      const double sq = __dmul_rn(dx, dx);
      acc = a == 0 ? sq : __dadd_rn(acc, sq);
      diff = a == dim ? dx : diff;
    }
    if (key_gt(wd, wi, acc, curr)) {
      heap_replace_root(hd, hi, k, acc, curr);
      wd = hd[0];
      wi = hi[0];
    }
    const uint32_t half = 1u << lc, room = lim - (uint32_t)curr;   // a child curr + s exists iff s < room
    const bool near_left = diff < 0.0;
    const uint32_t near_s = near_left ? half : 2u * half, far_s = near_left ? 2u * half : half;
    const float fb = fmaxf(__double2float_rd(__dmul_rn(diff, diff)), bound);
    const bool far_go = far_s < room && !((double)fb > wd);
    if (near_s < room) {
      if (far_go) { bnd[(lc + 1) * kKnnThreads] = fb; parked |= 2u << lc; }
      curr += (int32_t)near_s;
      ++lc;
    } else if (far_go) {                         // only the far child exists (it has the smaller index): no turn to remember
      curr += (int32_t)far_s;
      ++lc;
      bound = fb;
    } else {
      have = false;
    }
  }
  // nearest first: pop the heap from the back
  int32_t* out = nbr + (i - n0) * k;
  rad2[i] = (float)wd;     // squared neighbourhood radius: orders the points inside a batch (sort_keys_kernel)
  for (int m = k - 1; m >= 0; --m) {
    out[m] = hi[0];
    if (m > 0) {
      const double ld = hd[m * kKnnThreads];
      const int32_t li = hi[m * kKnnThreads];
      heap_replace_root(hd, hi, m, ld, li);
    }
  }
}

// ---- b3: depth ----------------------------------------------------------------------------------------
__global__ void max_depth_kernel(const int32_t* __restrict__ depth, int64_t n, unsigned long long* out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int32_t v = i < n ? depth[i] : 0;
  for (int o = 16; o > 0; o >>= 1) { int32_t w = __shfl_xor_sync(0xffffffffu, v, o); v = w > v ? w : v; }
  if ((threadIdx.x & 31) == 0 && v > 0) atomicMax(out, (unsigned long long)v);
}

// d_i = 1 + max_{j in c(i)} d_j.  The paper applies the update to all points in parallel until
// nothing changes: L sweeps of N k gathers.  The fixed point is unique, so it is reached here in ONE
// dataflow launch instead: depths start "pending" (-1, head 0), CTAs take chunks of the TREE order through a
// ticket, and a thread polls its k neighbours (all earlier in tree order, so held by a chunk that has started)
// until none is pending, then publishes its own depth.  The store sits inside the polling loop, so a neighbour
// that lives in the same warp makes progress without relying on independent thread scheduling.
__global__ void depth_init_kernel(int32_t* __restrict__ depth, int64_t n, int64_t n0) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) depth[i] = i < n0 ? 0 : -1;
}

__global__ void __launch_bounds__(256)
depth_flow_kernel(const int32_t* __restrict__ nbr, int64_t n, int64_t n0, int k, int32_t* depth,
                  unsigned long long* ticket, unsigned long long* timeout) {
  __shared__ unsigned long long s_chunk;
  if (threadIdx.x == 0) s_chunk = atomicAdd(ticket, 1ULL);
  __syncthreads();
  const int64_t i = n0 + (int64_t)s_chunk * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int32_t* row = nbr + (i - n0) * k;
  int32_t m = 0;
  int a = 0;
  bool done = false;
  unsigned spins = 0;
  const long long t0 = clock64();
  while (!done) {
    while (a < k) {
      int32_t dj;
      asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(dj) : "l"(depth + row[a]) : "memory");
      if (dj < 0) break;
      m = dj > m ? dj : m;
      ++a;
    }
    if (a == k) {
      asm volatile("st.relaxed.gpu.global.s32 [%0], %1;" ::"l"(depth + i), "r"(m + 1) : "memory");
      done = true;
    } else {
      if (++spins > 4) __nanosleep(spins > 64 ? 200 : 20);
      if ((spins & 1023u) == 0 && clock64() - t0 > 8000000000LL) {   // watchdog: a bug, never expected
        atomicAdd(timeout, 1ULL);
        asm volatile("st.relaxed.gpu.global.s32 [%0], %1;" ::"l"(depth + i), "r"(1) : "memory");
        done = true;
      }
    }
  }
}

// ---- b4: depth sort -----------------------------------------------------------------------------------
template <typename T>
__global__ void bbox_kernel(const T* __restrict__ x, int64_t n, int d, unsigned long long* bbox /*[2*kMaxD]*/) {
  // grid-stride partial extrema per thread, shuffle-reduced per warp, then one atomic pair per warp and dimension
  // (one atomic pair per POINT on six shared addresses was 50 ms of the 70 ms of this stage at N = 2^24)
  unsigned long long lo[kMaxD], hi[kMaxD];
#pragma unroll
  for (int t = 0; t < kMaxD; ++t) { lo[t] = ~0ULL; hi[t] = 0ULL; }
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
#pragma unroll
    for (int t = 0; t < kMaxD; ++t) {
      if (t < d) {
        const unsigned long long u = order_bits((double)x[i * d + t]);
        lo[t] = u < lo[t] ? u : lo[t];
        hi[t] = u > hi[t] ? u : hi[t];
      }
    }
  }
#pragma unroll
  for (int t = 0; t < kMaxD; ++t) {
    if (t < d) {
      for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long a = __shfl_xor_sync(0xffffffffu, lo[t], o), b = __shfl_xor_sync(0xffffffffu, hi[t], o);
        lo[t] = a < lo[t] ? a : lo[t];
        hi[t] = b > hi[t] ? b : hi[t];
      }
      if ((threadIdx.x & 31) == 0) { atomicMin(&bbox[2 * t], lo[t]); atomicMax(&bbox[2 * t + 1], hi[t]); }
    }
  }
}
__device__ __forceinline__ double unorder_bits(unsigned long long u) {
  u = (u & 0x8000000000000000ULL) ? (u & 0x7fffffffffffffffULL) : ~u;
  return __longlong_as_double((long long)u);
}

template <typename T>
__global__ void sort_keys_kernel(const T* __restrict__ x_tree, const int32_t* __restrict__ depth, int64_t n,
                                 int64_t n0, int d, int spatial, int cell_bits, int radius_bits, int depth_shift,
                                 const float* __restrict__ rad2, const unsigned long long* __restrict__ bbox,
                                 uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n - n0) return;
  int64_t i = n0 + e;
  uint64_t code = 0;
  if (spatial) {
    uint32_t cell[kMaxD];
    for (int t = 0; t < d; ++t) {
      double lo = unorder_bits(bbox[2 * t]), hi = unorder_bits(bbox[2 * t + 1]);
      double w = hi > lo ? hi - lo : 1.0;
      double f = ((double)x_tree[i * d + t] - lo) / w * (double)((uint64_t)1 << cell_bits);
      uint64_t c = f <= 0.0 ? 0 : (uint64_t)f;
      uint64_t cmax = ((uint64_t)1 << cell_bits) - 1;
      cell[t] = (uint32_t)(c > cmax ? cmax : c);
    }
    for (int b = 0; b < cell_bits; ++b)
      for (int t = 0; t < d; ++t) code |= (uint64_t)((cell[t] >> b) & 1u) << (b * d + t);
  }
  // optional neighbourhood-radius class (leading exponent bits of r^2), tight first: warps of a batch then hold
  // neighbourhoods of one scale; the Morton code orders the points inside a class.  Off by default: measured, it
  // halves the L1 hit rate of the gathers and nothing in the conditioning kernels depends on it.
  uint64_t rclass = 0;
  if (radius_bits > 0) rclass = (uint64_t)(__float_as_uint(rad2[i]) >> (31 - radius_bits)) & (((uint64_t)1 << radius_bits) - 1);
  keys[e] = ((uint64_t)depth[i] << depth_shift) | (rclass << (cell_bits * d)) | code;
  vals[e] = (uint32_t)i;
}

__global__ void positions_kernel(const uint32_t* __restrict__ sorted_tree, int64_t n, int64_t n0,
                                 uint32_t* __restrict__ pos2tree, uint32_t* __restrict__ tree2pos) {
  int64_t pos = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (pos >= n) return;
  uint32_t t = pos < n0 ? (uint32_t)pos : sorted_tree[pos - n0];
  pos2tree[pos] = t;
  tree2pos[t] = (uint32_t)pos;
}

template <typename T>
__global__ void emit_graph_kernel(const uint32_t* __restrict__ pos2tree, const uint32_t* __restrict__ tree2pos,
                                  const uint32_t* __restrict__ perm_tree, const T* __restrict__ x_tree,
                                  const int32_t* __restrict__ depth_tree, const int32_t* __restrict__ nbr_tree,
                                  int64_t n, int64_t n0, int d, int k, int64_t* __restrict__ perm,
                                  T* __restrict__ x_graph, int32_t* __restrict__ depth, int32_t* __restrict__ nbr,
                                  int64_t* __restrict__ boff) {
  int64_t pos = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (pos >= n) return;
  int64_t t = pos2tree[pos];
  perm[pos] = (int64_t)perm_tree[t];
  for (int a = 0; a < d; ++a) x_graph[pos * d + a] = x_tree[t * d + a];
  int32_t dep = depth_tree[t];
  depth[pos] = dep;
  if (pos >= n0) {
    const int32_t* src = nbr_tree + (t - n0) * k;
    int32_t* dst = nbr + (pos - n0) * k;
    for (int a = 0; a < k; ++a) dst[a] = (int32_t)tree2pos[src[a]];
    int32_t prev = pos == n0 ? 0 : depth_tree[pos2tree[pos - 1]];
    if (dep != prev) boff[dep - 1] = pos;       // first position of batch `dep` (depths are contiguous from 1)
    if (pos == n - 1) boff[dep] = n;
  }
}

}  // namespace gp

// ---- host driver ----------------------------------------------------------------------------------------
namespace gp {

static inline unsigned nblk(int64_t n, int t = 256) { return (unsigned)((n + t - 1) / t); }

template <typename KeyT>
static gp_status sort_pairs(void* tmp, size_t tmp_bytes, cub::DoubleBuffer<KeyT>& keys,
                            cub::DoubleBuffer<uint32_t>& vals, int64_t m, int begin_bit, int end_bit, cudaStream_t st) {
  if (m <= 0) return GP_OK;
  size_t need = 0;
  GP_CUDA_OK(cub::DeviceRadixSort::SortPairs(nullptr, need, keys, vals, (int)m, begin_bit, end_bit, st));
  if (need > tmp_bytes) return GP_ERR_WORKSPACE;
  GP_CUDA_OK(cub::DeviceRadixSort::SortPairs(tmp, need, keys, vals, (int)m, begin_bit, end_bit, st));
  count_launch(3);
  return GP_OK;
}

struct EventSet {
  cudaEvent_t ev[5];
  bool ok = true;
  EventSet() { for (auto& e : ev) if (cudaEventCreate(&e) != cudaSuccess) ok = false; }
  ~EventSet() { for (auto& e : ev) cudaEventDestroy(e); }
};

template <typename T>
static gp_status build_t(const T* x_user, int64_t n, int d, int k, int64_t n0, int dtype, int flags, int64_t* perm,
                         T* x_graph, int32_t* nbr, int32_t* depth, int64_t* boff_host, int max_batches,
                         int32_t* n_batches, char* ws, cudaStream_t st) {
  BuildLayout L = build_layout(n, d, k, dtype);
  Control* ctrl = (Control*)(ws + L.ctrl);
  uint32_t* rank = (uint32_t*)(ws + L.rank);
  uint64_t* keys_a = (uint64_t*)(ws + L.keys_a);
  uint64_t* keys_b = (uint64_t*)(ws + L.keys_b);
  uint32_t* vals_a = (uint32_t*)(ws + L.vals_a);
  uint32_t* vals_b = (uint32_t*)(ws + L.vals_b);
  uint32_t* seg = (uint32_t*)(ws + L.seg);
  uint32_t* perm_tree = (uint32_t*)(ws + L.perm_tree);
  T* x_tree = (T*)(ws + L.x_tree);
  int32_t* nbr_tree = (int32_t*)(ws + L.nbr_tree);
  int32_t* depth_tree = (int32_t*)(ws + L.depth_tree);
  uint32_t* tree2pos = (uint32_t*)(ws + L.tree2pos);
  uint32_t* pos2tree = (uint32_t*)(ws + L.pos2tree);
  unsigned long long* bbox = (unsigned long long*)(ws + L.bbox);
  int64_t* boff_dev = (int64_t*)(ws + L.boff);
  void* tmp = ws + L.cub_tmp;

  EventSet E;
  if (!E.ok) return GP_ERR_CUDA;
  GP_CUDA_OK(cudaMemsetAsync(ctrl, 0, kCtrlBytes, st));
  GP_CUDA_OK(cudaEventRecord(E.ev[0], st));

  // ---- b1: order -------------------------------------------------------------------------------------
  using CoordKey = typename std::conditional<sizeof(T) == 4, uint32_t, uint64_t>::type;
  const bool plain_order = (flags & GP_BUILD_PLAIN_ORDER) != 0;
  for (int dim = 0; dim < d; ++dim) {
    CoordKey* ck_a = (CoordKey*)keys_a;
    CoordKey* ck_b = (CoordKey*)keys_b;
    coord_keys_kernel<T, CoordKey><<<nblk(n), 256, 0, st>>>(x_user, n, d, dim, ck_a, vals_a);
    GP_LAUNCH_CHECK();
    cub::DoubleBuffer<CoordKey> kb(ck_a, ck_b);
    cub::DoubleBuffer<uint32_t> vb(vals_a, vals_b);
    GP_OK_OR_RETURN(sort_pairs<CoordKey>(tmp, L.cub_bytes, kb, vb, n, 0, (int)sizeof(CoordKey) * 8, st));
    if (plain_order) {
      scatter_rank_kernel<<<nblk(n), 256, 0, st>>>(vb.Current(), n, rank + (size_t)dim * n);
      GP_LAUNCH_CHECK();
    } else {   // the sorted ids ARE the level-0 list of this dimension
      GP_CUDA_OK(cudaMemcpyAsync(rank + (size_t)dim * n, vb.Current(), (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
    }
  }
  const TreeShape shape = tree_shape(n);
  if (!plain_order) {
    // lists: A in the rank region, B over keys_a + keys_b (contiguous: d * 4 n <= 16 n bytes)
    if (L.keys_b != L.keys_a + align_up((size_t)n * 8, 256) || L.vals_b != L.vals_a + align_up((size_t)n * 4, 256))
      return GP_ERR_WORKSPACE;
    uint32_t* la = rank;
    uint32_t* lb = (uint32_t*)keys_a;
    uint32_t* retired = vals_a;                  // where the partition drops the 2^l medians of a level (unused)
    int* n_sel = (int*)&ctrl->pad[0];            // its two counters (unused)
    uint32_t* side = seg;                        // 2 bits per id, all "left" to start with
    GP_CUDA_OK(cudaMemsetAsync(side, 0, ((size_t)n / 16 + 1) * 4, st));
    int64_t m = n;
    for (int l = 0; l <= shape.lam; ++l) {
      level_classify_kernel<<<nblk(m), 256, 0, st>>>(la + (size_t)(l % d) * n, m, l, shape, side, perm_tree);
      GP_LAUNCH_CHECK();
      if (l == shape.lam) break;                   // the last level: every remaining point is a node
      const int64_t n_left = subtree_prefix(shape, l + 1, (int64_t)1 << l);   // points in subtrees (l + 1, 0 .. 2^l - 1)
      for (int a = 0; a < d; ++a) {
        const uint32_t* in = la + (size_t)a * n;
        uint32_t* out = lb + (size_t)a * n;
        size_t need = 0;
        GP_CUDA_OK(cub::DevicePartition::If(nullptr, need, in, out, out + n_left, retired, n_sel, (int)m, SideIs{side, 0},
                                            SideIs{side, 1}, st));
        if (need > L.cub_bytes) return GP_ERR_WORKSPACE;
        GP_CUDA_OK(cub::DevicePartition::If(tmp, need, in, out, out + n_left, retired, n_sel, (int)m, SideIs{side, 0},
                                            SideIs{side, 1}, st));
        count_launch(2);
      }
      uint32_t* t_ = la; la = lb; lb = t_;
      m -= (int64_t)1 << l;
    }
  } else {
  int rank_bits = 1;
  while (((int64_t)1 << rank_bits) < n) ++rank_bits;
  {
    cub::DoubleBuffer<uint64_t> kb(keys_a, keys_b);
    cub::DoubleBuffer<uint32_t> vb(vals_a, vals_b);
    iota_seg_kernel<<<nblk(n), 256, 0, st>>>(vb.Current(), seg, n);
    GP_LAUNCH_CHECK();
    int64_t m_sort = n;
    for (int l = 0; l <= shape.lam; ++l) {
      // elements retired at level l-1 carry segment id 2^l and sink behind the active ones in this sort
      level_keys_kernel<<<nblk(m_sort), 256, 0, st>>>(vb.Current(), seg, rank + (size_t)(l % d) * n, m_sort,
                                                      rank_bits, kb.Current());
      GP_LAUNCH_CHECK();
      GP_OK_OR_RETURN(sort_pairs<uint64_t>(tmp, L.cub_bytes, kb, vb, m_sort, 0, rank_bits + l + 1, st));
      int64_t m_active = l == 0 ? n : m_sort - ((int64_t)1 << (l - 1));
      level_split_kernel<<<nblk(m_active), 256, 0, st>>>(kb.Current(), vb.Current(), m_active, rank_bits, l, shape,
                                                         seg, perm_tree);
      GP_LAUNCH_CHECK();
      m_sort = m_active;
    }
  }
  }
  gather_points_kernel<T><<<nblk(n), 256, 0, st>>>(x_user, perm_tree, n, d, x_tree);
  GP_LAUNCH_CHECK();
  GP_CUDA_OK(cudaEventRecord(E.ev[1], st));

  // ---- b2: preceding kNN -----------------------------------------------------------------------------
  if (n > n0) {
    int64_t n_threads = ((int64_t)2 << shape.lam) - 1;
    unsigned long long* ovf = &ctrl->n_bad;      // zeroed above; read back with the depth watchdog below
    float* rad2 = (float*)seg;                   // the segment ids of b1 are dead: reuse the buffer (tree order)
    const bool plain = (flags & GP_BUILD_PLAIN_KNN) != 0;
    const int nlev = shape.lam + 2;                // levels 0 .. lam + 1 can be indexed (level 0 is never parked)
    const size_t sm_bytes = (size_t)kKnnThreads * (12 * (size_t)k + 4 * (size_t)nlev);
    if (!plain && d <= 3 && sm_bytes <= 200 * 1024) {
      // fp32: the order stage's key buffers (16 n bytes, contiguous, checked there) are dead until the depth sort
      const float4* x4 = nullptr;
      // (only once the coordinates no longer fit the L2: measured 975 -> 881 ms at N = 2^28, 209 -> 202 ms at 2^26,
      // and 61 -> 62 ms at 2^24, where the extra pass is all it adds)
      if (sizeof(T) == 4 && (size_t)n * d * 4 > ((size_t)96 << 20) && L.keys_b == L.keys_a + align_up((size_t)n * 8, 256)) {
        pack_points4_kernel<<<nblk(n), 256, 0, st>>>((const float*)x_tree, n, d, (float4*)keys_a);
        GP_LAUNCH_CHECK();
        x4 = (const float4*)keys_a;
      }
#define GP_KNN_SM2(DD, P4) { \
      GP_CUDA_OK(cudaFuncSetAttribute(knn_sm_kernel<T, DD, P4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)); \
      knn_sm_kernel<T, DD, P4><<<nblk(n_threads, kKnnThreads), kKnnThreads, sm_bytes, st>>>(x_tree, x4, n, n0, k, nlev, n_threads, nbr_tree, rad2); }
#define GP_KNN_SM(DD) { if (x4) GP_KNN_SM2(DD, true) else GP_KNN_SM2(DD, false) }
      if (d == 1) GP_KNN_SM(1) else if (d == 2) GP_KNN_SM(2) else GP_KNN_SM(3)
#undef GP_KNN_SM2
#undef GP_KNN_SM
    }
    else if (k <= 16) knn_kernel<T, 16><<<nblk(n_threads, 128), 128, 0, st>>>(x_tree, n, n0, d, k, n_threads, nbr_tree, rad2, ovf);
    else if (k <= 32) knn_kernel<T, 32><<<nblk(n_threads, 128), 128, 0, st>>>(x_tree, n, n0, d, k, n_threads, nbr_tree, rad2, ovf);
    else if (k <= 64) knn_kernel<T, 64><<<nblk(n_threads, 128), 128, 0, st>>>(x_tree, n, n0, d, k, n_threads, nbr_tree, rad2, ovf);
    else knn_kernel<T, 128><<<nblk(n_threads, 128), 128, 0, st>>>(x_tree, n, n0, d, k, n_threads, nbr_tree, rad2, ovf);
    GP_LAUNCH_CHECK();
  }
  GP_CUDA_OK(cudaEventRecord(E.ev[2], st));

  // ---- b3: depth fixed point --------------------------------------------------------------
  depth_init_kernel<<<nblk(n), 256, 0, st>>>(depth_tree, n, n0);
  GP_LAUNCH_CHECK();
  int64_t max_depth = 0;
  if (n > n0) {
    GP_CUDA_OK(cudaMemsetAsync(&ctrl->ticket, 0, 8, st));
    GP_CUDA_OK(cudaMemsetAsync(&ctrl->timeout, 0, 8, st));
    depth_flow_kernel<<<nblk(n - n0), 256, 0, st>>>(nbr_tree, n, n0, k, depth_tree, &ctrl->ticket, &ctrl->timeout);
    GP_LAUNCH_CHECK();
    GP_CUDA_OK(cudaMemsetAsync(&ctrl->ticket, 0, 8, st));
    unsigned long long* mx = &ctrl->ticket;
    max_depth_kernel<<<nblk(n), 256, 0, st>>>(depth_tree, n, mx);
    GP_LAUNCH_CHECK();
    unsigned long long h = 0;
    GP_CUDA_OK(cudaMemcpyAsync(&h, mx, 8, cudaMemcpyDeviceToHost, st));
    GP_CUDA_OK(cudaStreamSynchronize(st));
    max_depth = (int64_t)h;
    unsigned long long stuck = 0;
    GP_CUDA_OK(cudaMemcpy(&stuck, &ctrl->timeout, 8, cudaMemcpyDeviceToHost));
    if (stuck) return GP_ERR_CUDA;                // the depth dataflow's watchdog fired
    unsigned long long dropped = 0;
    GP_CUDA_OK(cudaMemcpy(&dropped, &ctrl->n_bad, 8, cudaMemcpyDeviceToHost));
    if (dropped) return GP_ERR_UNSUPPORTED;       // a kNN walk ran out of stack: the graph would be wrong
    if (max_depth > max_batches || max_depth > kMaxBatches) return GP_ERR_INVALID_ARG;
  }
  GP_CUDA_OK(cudaEventRecord(E.ev[3], st));

  // ---- b4: depth sort, remap ---------------------------------------------------------------------------
  if (n > n0) {
    int depth_bits = 1;
    while (((int64_t)1 << depth_bits) <= max_depth) ++depth_bits;
    const int spatial = (flags & GP_BUILD_SPATIAL_BATCHES) ? 1 : 0;
    const int radius_bits = (flags & GP_BUILD_RADIUS_CLASSES) ? 6 : 0;   // exponent of r^2 / 4: one class per two octaves of r
    int cell_bits = 0, depth_shift = radius_bits;
    if (spatial) {
      cell_bits = (63 - depth_bits - radius_bits) / d;
      if (cell_bits > 21) cell_bits = 21;
      depth_shift = cell_bits * d + radius_bits;
      GP_CUDA_OK(cudaMemsetAsync(bbox, 0xff, 8 * 2 * kMaxD, st));
      for (int t = 0; t < d; ++t) GP_CUDA_OK(cudaMemsetAsync(bbox + 2 * t + 1, 0, 8, st));
      bbox_kernel<T><<<nblk(n) < 148u * 8u ? nblk(n) : 148u * 8u, 256, 0, st>>>(x_tree, n, d, bbox);
      GP_LAUNCH_CHECK();
    }
    cub::DoubleBuffer<uint64_t> kb(keys_a, keys_b);
    cub::DoubleBuffer<uint32_t> vb(vals_a, vals_b);
    sort_keys_kernel<T><<<nblk(n - n0), 256, 0, st>>>(x_tree, depth_tree, n, n0, d, spatial, cell_bits, radius_bits,
                                                      depth_shift, (const float*)seg, bbox, kb.Current(), vb.Current());
    GP_LAUNCH_CHECK();
    GP_OK_OR_RETURN(sort_pairs<uint64_t>(tmp, L.cub_bytes, kb, vb, n - n0, 0, depth_shift + depth_bits, st));
    positions_kernel<<<nblk(n), 256, 0, st>>>(vb.Current(), n, n0, pos2tree, tree2pos);
    GP_LAUNCH_CHECK();
  } else {
    positions_kernel<<<nblk(n), 256, 0, st>>>(nullptr, n, n0, pos2tree, tree2pos);
    GP_LAUNCH_CHECK();
  }
  emit_graph_kernel<T><<<nblk(n), 256, 0, st>>>(pos2tree, tree2pos, perm_tree, x_tree, depth_tree, nbr_tree, n, n0, d, k,
                                                perm, x_graph, depth, nbr, boff_dev);
  GP_LAUNCH_CHECK();
  GP_CUDA_OK(cudaEventRecord(E.ev[4], st));
  if (max_depth > 0)
    GP_CUDA_OK(cudaMemcpyAsync(boff_host, boff_dev, (size_t)(max_depth + 1) * 8, cudaMemcpyDeviceToHost, st));
  GP_CUDA_OK(cudaStreamSynchronize(st));
  if (max_depth == 0) boff_host[0] = n0;
  *n_batches = (int32_t)max_depth;
  Control h{};
  for (int s = 0; s < 4; ++s) {
    float ms = 0.f;
    GP_CUDA_OK(cudaEventElapsedTime(&ms, E.ev[s], E.ev[s + 1]));
    h.build_ms[s] = ms;
  }
  GP_CUDA_OK(cudaMemcpy(ctrl->build_ms, h.build_ms, sizeof(h.build_ms), cudaMemcpyHostToDevice));
  return GP_OK;
}
}  // namespace gp

using namespace gp;

extern "C" {

size_t gp_graph_build_workspace_bytes(int64_t n, int32_t d, int32_t k, int32_t dtype) {
  if (n <= 0 || d < 1 || d > kMaxD || k < 1 || k > kMaxK || (dtype != GP_F32 && dtype != GP_F64)) return 0;
  return build_layout(n, d, k, dtype).total;
}

gp_status gp_graph_build(const void* x_user, int64_t n, int32_t d, int32_t k, int64_t n0, int32_t dtype,
                         int32_t build_flags, int64_t* perm, void* x_graph, int32_t* nbr, int32_t* depth,
                         int64_t* batch_off_host, int32_t max_batches, int32_t* n_batches, void* ws, size_t ws_bytes,
                         void* cuda_stream) {
  if (!x_user || !perm || !x_graph || !depth || !batch_off_host || !n_batches) return GP_ERR_INVALID_ARG;
  if (n <= 0 || n0 < 0 || n0 > n || d < 1 || k < 1 || max_batches < 1) return GP_ERR_INVALID_ARG;
  if (d > kMaxD || k > kMaxK || n >= (1LL << 31)) return GP_ERR_UNSUPPORTED;
  if (dtype != GP_F32 && dtype != GP_F64) return GP_ERR_INVALID_ARG;
  if (n0 < k && n0 < n) return GP_ERR_INVALID_ARG;
  if (n > n0 && !nbr) return GP_ERR_INVALID_ARG;
  size_t need = gp_graph_build_workspace_bytes(n, d, k, dtype);
  if (!ws || ws_bytes < need || (((uintptr_t)ws) & 255) != 0) return GP_ERR_WORKSPACE;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return GP_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (dtype == GP_F64)
    return build_t<double>((const double*)x_user, n, d, k, n0, dtype, build_flags, perm, (double*)x_graph, nbr, depth,
                           batch_off_host, max_batches, n_batches, (char*)ws, st);
  return build_t<float>((const float*)x_user, n, d, k, n0, dtype, build_flags, perm, (float*)x_graph, nbr, depth,
                        batch_off_host, max_batches, n_batches, (char*)ws, st);
}

gp_status gp_graph_build_times(void* ws, double* ms4_host) {
  if (!ws || !ms4_host) return GP_ERR_INVALID_ARG;
  Control h;
  GP_CUDA_OK(cudaMemcpy(&h, ws, sizeof(Control), cudaMemcpyDeviceToHost));
  for (int s = 0; s < 4; ++s) ms4_host[s] = h.build_ms[s];
  return GP_OK;
}

}  // extern "C"
