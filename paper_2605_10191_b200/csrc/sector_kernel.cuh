// Device code of the sector sweep (sector.cuh).  Included by the sector_m*.cu instantiation files
// (one tile size M each, so that they compile in parallel).
#pragma once

#include <type_traits>
#include <utility>

#include "sector.cuh"

namespace polfed {
namespace sector {

enum { MODE_STEP = 0, MODE_INIT = 1, MODE_LAST = 2 };

struct SecArgs {
  long long n;
  int n_tiles, n_panels;
  const int32_t* tile_row0;
  const int32_t* tile_class;
  const uint16_t* units;
  const uint4* meta;       // [n][2]
  const int32_t* dst_nat;  // MODE_LAST: position -> caller's row
  double ccoef[kTileMaxCrossCoef + 1];
  double t1, t2;
  const double* X1;  // b_{k+1}, panel-major [s/8][n][8], this layout
  const double* Pk;  // partial b_k
  const double* V;
  double* Bout;      // b_k, other layout
  double* Pout;      // partial b_{k-1}, other layout
  double* W;         // MODE_LAST: n x w_ld row-major, caller's row order
  int w_ld;
  int* counter;      // work-item counter of this sweep (zero on entry)
  double cK, pf, ps, qs, rs, cs;
  unsigned buf_bytes;  // bytes of one shared-memory tile buffer
  SectorTables tab;
};

// ---- compile-time combinatorics --------------------------------------------------------------
constexpr int cx_binom(int n, int k) {
  if (k < 0 || k > n) return 0;
  int r = 1;
  for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
  return r;
}
constexpr int cx_popc(unsigned c) {
  int n = 0;
  for (; c; c >>= 1) n += (int)(c & 1u);
  return n;
}
// r-th G-bit integer with J set bits, ascending (= the order of basis states, R12)
constexpr unsigned cx_cfg(int G, int J, int r) {
  int cnt = 0;
  for (unsigned c = 0; c < (1u << G); ++c)
    if (cx_popc(c) == J) {
      if (cnt == r) return c;
      ++cnt;
    }
  return 0u;
}
constexpr int cx_rank(unsigned c) {
  const int J = cx_popc(c);
  int cnt = 0;
  for (unsigned d = 0; d < c; ++d)
    if (cx_popc(d) == J) ++cnt;
  return cnt;
}

template <class F, int... R>
__device__ __forceinline__ void static_for(F&& f, std::integer_sequence<int, R...>) {
  (f(std::integral_constant<int, R>{}), ...);
}

// Row R of the hop operator of a group of G sites in the sector of J particles: all bonds
// (A, A+1) with amplitude t1 and (A, A+2) with amplitude t2 (sign (-1)^{n_{A+1}} if JW).
template <int G, int J, bool NNN, bool JW, int R, int N>
struct RowOp {
  static constexpr unsigned c = cx_cfg(G, J, R);
  template <int A>
  static __device__ __forceinline__ void nn(const double (&x)[N], double t1, double& acc) {
    if constexpr (A + 1 < G) {
      if constexpr ((((c >> A) ^ (c >> (A + 1))) & 1u) != 0u) {
        constexpr int r2 = cx_rank(c ^ (3u << A));
        acc = fma(t1, x[r2], acc);
      }
    }
  }
  template <int A>
  static __device__ __forceinline__ void nnn(const double (&x)[N], double t2, double& acc) {
    if constexpr (NNN && A + 2 < G) {
      if constexpr ((((c >> A) ^ (c >> (A + 2))) & 1u) != 0u) {
        constexpr int r2 = cx_rank(c ^ (5u << A));
        if constexpr (JW && ((c >> (A + 1)) & 1u) != 0u)
          acc = fma(-t2, x[r2], acc);
        else
          acc = fma(t2, x[r2], acc);
      }
    }
  }
  template <int... A>
  static __device__ __forceinline__ double apply(const double (&x)[N], double t1, double t2,
                                                 double acc, std::integer_sequence<int, A...>) {
    double acc2 = 0.0;  // two chains: the bonds (A, A+1) and (A, A+2)
    (nn<A>(x, t1, acc), ...);
    (nnn<A>(x, t2, acc2), ...);
    if constexpr (NNN) acc += acc2;
    return acc;
  }
};

template <int G, int J, bool NNN, bool JW, int R, int N>
__device__ __forceinline__ double group_row(const double (&x)[N], double t1, double t2, double acc) {
  return RowOp<G, J, NNN, JW, R, N>::apply(x, t1, t2, acc, std::make_integer_sequence<int, G>{});
}

// ---- memory helpers -----------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
// shared-memory reads that the compiler may move across the (disjoint) stores of other rows
// (no memory clobber); `epoch` changes at every CTA barrier, so that two reads of one address on
// different sides of a barrier are never merged
__device__ __forceinline__ double lds64(uint32_t addr, uint32_t epoch) {
  double v;
  asm("ld.shared.f64 %0, [%1];  // %2" : "=d"(v) : "r"(addr), "r"(epoch));
  return v;
}
__device__ __forceinline__ void sts64(uint32_t addr, double v) {
  asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ double ldg64_stream(const double* p, uint64_t pol) {  // touched once
  double v;
  asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ double ldg64_l2(const double* p) {  // re-read from L2, not kept in L1
  double v;
  asm("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ uint4 ldg128(const uint4* p) {
  uint4 v;
  asm("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ void stg64_stream(double* p, double v, uint64_t pol) {
  asm volatile("st.global.L1::no_allocate.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, unsigned bytes, uint64_t* bar,
                                         uint64_t pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], "
      "%2, [%3], %4;" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "SEC_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra SEC_DONE;\n"
      "bra SEC_WAIT;\n"
      "SEC_DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async;" ::: "memory");
}

__device__ __forceinline__ double signed_coef(double cf, uint32_t sign_bit31) {
  return __hiloint2double(__double2hiint(cf) ^ (int)(sign_bit31 & 0x80000000u), __double2loint(cf));
}
constexpr uint32_t kPosMask = (1u << kCrossPosBits) - 1u;

// Predicated 16-byte reads: lanes whose predicate is off issue no access and get zeros.
__device__ __forceinline__ double2 lds128(uint32_t addr, uint32_t epoch) {
  double2 v;
  asm("ld.shared.v2.f64 {%0,%1}, [%2];  // %3" : "=d"(v.x), "=d"(v.y) : "r"(addr), "r"(epoch));
  return v;
}
__device__ __forceinline__ double2 lds128_if(uint32_t addr, uint32_t on, uint32_t epoch) {
  double2 v;
  asm("{\n.reg .pred q;\nsetp.ne.u32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\n"
      "mov.f64 %1, 0d0000000000000000;\n@q ld.shared.v2.f64 {%0,%1}, [%2];  // %4\n}"
      : "=d"(v.x), "=d"(v.y)
      : "r"(addr), "r"(on), "r"(epoch));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, double2 v) {
  asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ double2 ldg128_stream(const double* p, uint64_t pol) {
  double2 v;
  asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
      : "=d"(v.x), "=d"(v.y)
      : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ double2 ldg128_l2_if(const double* p, uint32_t on) {
  double2 v;
  asm("{\n.reg .pred q;\nsetp.ne.u32 q, %3, 0;\nmov.f64 %0, 0d0000000000000000;\n"
      "mov.f64 %1, 0d0000000000000000;\n@q ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];\n}"
      : "=d"(v.x), "=d"(v.y)
      : "l"(p), "r"(on));
  return v;
}
__device__ __forceinline__ void stg128_stream(double* p, double2 v, uint64_t pol) {
  asm volatile("st.global.L1::no_allocate.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" ::"l"(p),
               "d"(v.x), "d"(v.y), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void fma2(double c, const double2 x, double2& acc) {
  acc.x = fma(c, x.x, acc.x);
  acc.y = fma(c, x.y, acc.y);
}

// ---- view 1: a G1-fibre (n1 consecutive rows) in registers ----------------------------------
//   dst[r] = alpha (O_G1 src)[r] + beta src[r] + gamma dst[r]       (gamma term only if use_old)
// at1 = alpha t1, at2 = alpha t2.  Addresses include the lane's 8-byte column offset.
template <int G, int J, bool NNN, bool JW>
__device__ __forceinline__ void view1_unit(uint32_t src, uint32_t dst, double at1, double at2,
                                           double beta, double gamma, bool use_old,
                                           uint32_t epoch) {
  constexpr int N = cx_binom(G, J);
  double x[N];
  static_for([&](auto rc) {
    constexpr int R = decltype(rc)::value;
    x[R] = lds64(src + R * 64, epoch);
  }, std::make_integer_sequence<int, N>{});
  if (use_old) {
    static_for([&](auto rc) {
      constexpr int R = decltype(rc)::value;
      const double acc = fma(gamma, lds64(dst + R * 64, epoch), beta * x[R]);
      sts64(dst + R * 64, group_row<G, J, NNN, JW, R, N>(x, at1, at2, acc));
    }, std::make_integer_sequence<int, N>{});
  } else {
    static_for([&](auto rc) {
      constexpr int R = decltype(rc)::value;
      sts64(dst + R * 64, group_row<G, J, NNN, JW, R, N>(x, at1, at2, beta * x[R]));
    }, std::make_integer_sequence<int, N>{});
  }
}

// ---- view 2: a G2-fibre (n2 rows, pitch `pitch` bytes) in registers -------------------------
//   dst[r] += alpha (O_G2 src)[r]
template <int G, int J, bool NNN, bool JW>
__device__ __forceinline__ void view2_unit(uint32_t src, uint32_t dst, uint32_t pitch, double at1,
                                           double at2, uint32_t epoch) {
  constexpr int N = cx_binom(G, J);
  double x[N];
  static_for([&](auto rc) {
    constexpr int R = decltype(rc)::value;
    x[R] = lds64(src + R * pitch, epoch);
  }, std::make_integer_sequence<int, N>{});
  static_for([&](auto rc) {
    constexpr int R = decltype(rc)::value;
    const double acc = lds64(dst + R * pitch, epoch);
    sts64(dst + R * pitch, group_row<G, J, NNN, JW, R, N>(x, at1, at2, acc));
  }, std::make_integer_sequence<int, N>{});
}

template <int G, bool NNN, bool JW, int... J>
__device__ __forceinline__ void view1_dispatch(int j, uint32_t src, uint32_t dst, double at1,
                                               double at2, double beta, double gamma, bool use_old,
                                               uint32_t epoch, std::integer_sequence<int, J...>) {
  ((j == J ? (view1_unit<G, J, NNN, JW>(src, dst, at1, at2, beta, gamma, use_old, epoch), 0) : 0),
   ...);
}
template <int G, bool NNN, bool JW, int... J>
__device__ __forceinline__ void view2_dispatch(int j, uint32_t src, uint32_t dst, uint32_t pitch,
                                               double at1, double at2, uint32_t epoch,
                                               std::integer_sequence<int, J...>) {
  ((j == J ? (view2_unit<G, J, NNN, JW>(src, dst, pitch, at1, at2, epoch), 0) : 0), ...);
}

__device__ __forceinline__ int claim(int* counter, int step, int lane) {
  int v = 0;
  if (lane == 0) v = atomicAdd(counter, step);
  return __shfl_sync(0xffffffffu, v, 0);
}

// The structured part of one phase: dst = alpha O_l src + beta src (+ gamma dst), O_l = O_G1 + O_G2,
// in two steps (all warps of the CTA), each followed by a CTA barrier.
template <int G1, bool NNN, bool JW>
__device__ __forceinline__ void structured_v1(const SecArgs& a, int k, const uint16_t* units1, int* ctr,
                                              uint32_t src, uint32_t dst, double alpha, double beta,
                                              double gamma, bool use_old, uint32_t& epoch, int lane) {
  const int grp = lane >> 3;
  const double at1 = alpha * a.t1, at2 = alpha * a.t2;
  const int nu1 = a.tab.n_units[0][k];
  for (int u = claim(ctr, 1, lane); u < nu1; u = claim(ctr, 1, lane)) {
    const int unit = units1[u], j1 = unit & 7, i2 = (unit >> 3) * kSecGroups + grp;
    if (i2 < a.tab.n2[k - j1]) {
      const uint32_t off = (uint32_t)(a.tab.srow[k][j1] + i2 * a.tab.n1p[j1]) * 64u;
      view1_dispatch<G1, NNN, JW>(j1, src + off, dst + off, at1, at2, beta, gamma, use_old, epoch,
                                  std::make_integer_sequence<int, G1 + 1>{});
    }
  }
  __syncthreads();
  ++epoch;
}
template <int G2, bool NNN, bool JW>
__device__ __forceinline__ void structured_v2(const SecArgs& a, int k, const uint16_t* units2, int* ctr,
                                              uint32_t src, uint32_t dst, double alpha,
                                              uint32_t& epoch, int lane) {
  const int grp = lane >> 3;
  const double at1 = alpha * a.t1, at2 = alpha * a.t2;
  const int nu2 = a.tab.n_units[1][k];
  for (int u = claim(ctr, 1, lane); u < nu2; u = claim(ctr, 1, lane)) {
    const int unit = units2[u], j1 = unit & 7, i1 = (unit >> 3) * kSecGroups + grp;
    if (i1 < a.tab.n1[j1]) {
      const uint32_t off = (uint32_t)(a.tab.srow[k][j1] + i1) * 64u;
      view2_dispatch<G2, NNN, JW>(k - j1, src + off, dst + off, (uint32_t)a.tab.n1p[j1] * 64u, at1,
                                  at2, epoch, std::make_integer_sequence<int, G2 + 1>{});
    }
  }
  __syncthreads();
  ++epoch;
}

// Row record (sector.cuh): word 0 other-layout position, words 1-2 three cross-group entries and
// (bits 16-31 of word 2) the row's own shared-memory row, word 3 and words 4-5 cross-cut words,
// words 6-7 the diagonal.
struct RowMeta {
  uint4 m0, m1;
};
__device__ __forceinline__ RowMeta load_meta(const uint4* meta, int pos, int nrows, bool both) {
  RowMeta r;
  r.m0 = make_uint4(0u, 0u, 0u, kCrossNone);
  r.m1 = make_uint4(kCrossNone, kCrossNone, 0u, 0u);
  if (pos < nrows) {
    r.m0 = ldg128(meta + (size_t)pos * 2);
    if (both) r.m1 = ldg128(meta + (size_t)pos * 2 + 1);
  }
  return r;
}

// The global operands of a row of the phase-2 row pass: its cross-cut partners.
struct RowOperands {
  double2 h0, h1, h2;
};
__device__ __forceinline__ double2 load_stream_if(const double* rows, int pos, int nrows, bool on,
                                                  uint64_t pol) {
  double2 v = make_double2(0.0, 0.0);
  if (on && pos < nrows) v = ldg128_stream(rows + (size_t)pos * kSecPanel, pol);
  return v;
}
__device__ __forceinline__ RowOperands load_operands(const RowMeta& m, const double* X1) {
  RowOperands o;
  const uint32_t c0 = m.m0.w, c1 = m.m1.x, c2 = m.m1.y;
  o.h0 = ldg128_l2_if(X1 + (size_t)(c0 & kPosMask) * kSecPanel, c0 != kCrossNone);
  o.h1 = ldg128_l2_if(X1 + (size_t)(c1 & kPosMask) * kSecPanel, c1 != kCrossNone);
  o.h2 = ldg128_l2_if(X1 + (size_t)(c2 & kPosMask) * kSecPanel, c2 != kCrossNone);
  return o;
}

// Cross-group partners of a row: entry slots 0..2 carry t1, t2, t2 (sector.cuh).
__device__ __forceinline__ void cross_group(const RowMeta& m, uint32_t s_tile, double t1, double t2,
                                            uint32_t epoch, double2& acc) {
  const uint32_t e0 = m.m0.y & 0xffffu, e1 = m.m0.y >> 16, e2 = m.m0.z & 0xffffu;
  const double2 g0 = lds128_if(s_tile + (e0 & kXgRow) * 64u, e0 & kXgValid, epoch);
  const double2 g1 = lds128_if(s_tile + (e1 & kXgRow) * 64u, e1 & kXgValid, epoch);
  const double2 g2 = lds128_if(s_tile + (e2 & kXgRow) * 64u, e2 & kXgValid, epoch);
  fma2(signed_coef(t1, e0 << 18), g0, acc);
  fma2(signed_coef(t2, e1 << 18), g1, acc);
  fma2(signed_coef(t2, e2 << 18), g2, acc);
}

// Ask L2 for `bytes` (a multiple of 16) at p, 2 KB per participating thread starting at thread t0.
__device__ __forceinline__ void l2_prefetch(const void* p, unsigned bytes, int tid, int t0) {
  const unsigned at = (unsigned)(tid - t0) * 2048u;
  if (tid >= t0 && at < bytes)
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(static_cast<const char*>(p) + at),
                 "r"(min(2048u, bytes - at))
                 : "memory");
}

constexpr int kTailRows = 8;  // rows per warp iteration of the row passes: 4 lanes x 16 bytes each
constexpr int kSecWarps = kSecThreads / 32;
constexpr int kBatch = 3;  // row passes: 8-row groups per warp and batch

template <int M, bool NNN, bool JW, int MODE>
__global__ void __launch_bounds__(kSecThreads, 1) sector_sweep_kernel(const SecArgs a) {
  constexpr int G1 = sector_g1(M), G2 = M - G1;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ uint64_t bar;
  __shared__ int4 s_work[2];  // work item, first row, rows, class of the tile
  __shared__ uint16_t s_units[2 * (M + 1) * kSecMaxUnits];
  // work counters per tile (view 1, view 2, row pass of phase 2; the same of phase 3), one set per
  // tile parity: a tile zeroes the other set, so no barrier is needed at the top of a tile
  __shared__ int s_ctr_all[2][6];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int l8 = lane & 7;                   // structured passes: 8 lanes x 8 bytes per row
  const int q = lane & 3, slot = lane >> 2;  // row passes: 4 lanes x 16 bytes per row
  const int total = a.n_tiles * a.n_panels;
  auto next_work = [&]() {  // one thread: claim a work item and look its tile up
    int4 w = make_int4(atomicAdd(a.counter, 1), 0, 0, 0);
    if (w.x < total) {
      const int tile = w.x / a.n_panels;
      w.y = __ldg(a.tile_row0 + tile);
      w.z = __ldg(a.tile_row0 + tile + 1) - w.y;
      w.w = __ldg(a.tile_class + tile);
    }
    return w;
  };
  for (int i = tid; i < 2 * (M + 1) * kSecMaxUnits; i += kSecThreads) s_units[i] = a.units[i];
  if (tid < 12) s_ctr_all[tid / 6][tid % 6] = 0;
  if (tid == 0) {
    mbar_init(&bar, 1);
    s_work[0] = next_work();
  }
  __syncthreads();
  unsigned parity = 0;
  uint32_t epoch = 0;
  const size_t panel_stride = (size_t)a.n * kSecPanel;
  const uint64_t pol_first = policy_evict_first(), pol_last = policy_evict_last();
  const uint32_t sA = smem_u32(smem_raw), sB = sA + a.buf_bytes;

  for (int it = 0;; ++it) {
    // work items in tile-major order: the s/8 panels of a tile are consecutive items, so they run at
    // about the same time on different SMs and share the tile's row records in L2
    const int4 wi = s_work[it & 1];
    const int work = wi.x, row0 = wi.y, nrows = wi.z, k = wi.w;
    if (work >= total) break;
    const int panel = work % a.n_panels;
    int* const s_ctr = s_ctr_all[it & 1];
    if (tid < 6) s_ctr_all[(it + 1) & 1][tid] = 0;
    if (MODE != MODE_INIT && warp == 0) {
      // the tile panels of b_{k+1} -> buffer A and of the partial b_k -> buffer B: one bulk copy
      // each, or one per fibre when the fibre pitch is padded
      if (lane == 0) {
        fence_proxy_async();
        mbar_expect_tx(&bar, 2u * (unsigned)nrows * 64u);
      }
      __syncwarp();
      const size_t off = panel * panel_stride + (size_t)row0 * kSecPanel;
      if (a.tab.rows_p[k] == nrows) {  // no padding: the whole tile is one run
        if (lane < 2)
          bulk_g2s(lane ? sB : sA, (lane ? a.Pk : a.X1) + off, (unsigned)nrows * 64u, &bar, lane ? pol_first : pol_last);
      } else {
        const int j_lo = k > G2 ? k - G2 : 0, j_hi = k < G1 ? k : G1;
        for (int j1 = j_lo; j1 <= j_hi; ++j1) {
          const int n1 = a.tab.n1[j1], n1p = a.tab.n1p[j1], n2 = a.tab.n2[k - j1];
          const int p0 = a.tab.sbase[k][j1], r0 = a.tab.srow[k][j1];
          for (int i = lane; i < 2 * n2; i += 32) {
            const int i2 = i >> 1;
            const double* src = ((i & 1) ? a.Pk : a.X1) + off + (size_t)(p0 + i2 * n1) * kSecPanel;
            bulk_g2s(((i & 1) ? sB : sA) + (unsigned)(r0 + i2 * n1p) * 64u, src, (unsigned)n1 * 64u,
                     &bar, (i & 1) ? pol_first : pol_last);
          }
        }
      }
    }
    const uint4* meta = a.meta + (size_t)row0 * 2;
    const double* X1 = a.X1 + panel * panel_stride + 2 * q;
    const double* V = a.V + panel * panel_stride + (size_t)row0 * kSecPanel + 2 * q;
    double* Bout = a.Bout + panel * panel_stride + 2 * q;
    double* Pout = a.Pout + panel * panel_stride + 2 * q;
    const uint16_t* units1 = s_units + k * kSecMaxUnits;
    const uint16_t* units2 = s_units + (M + 1 + k) * kSecMaxUnits;
    // MODE_INIT: rows dealt out statically, 8 per warp and turn
    const int pos0 = warp * kTailRows + slot;
    constexpr int kStride = kSecWarps * kTailRows;
    // The next work item is claimed by the last warp (only its lane 0 waits for the atomic) and
    // read after later barriers.
    if (tid == kSecThreads - 32) s_work[(it + 1) & 1] = next_work();

    // phase 2: B (= P_k) += pf O_l b_{k+1}, then b_k = B + pf (D b_{k+1} + cross terms)
    // phase 3: A = ps O_l b_k + qs b_k + rs b_{k+1}, then P_{k-1} = A + ps cross-group + cs V
    // (one loop, so that the structured passes are instantiated once)
#pragma unroll 1
    for (int ph = 2; ph <= (MODE == MODE_LAST ? 2 : 3); ++ph) {
      if (MODE == MODE_INIT && ph == 2) {
        // ---- b_K = c_K V -> other layout and buffer B -----------------------------------------
        for (int pos = pos0; pos < nrows; pos += kStride) {
          const uint4 m0 = ldg128(meta + (size_t)pos * 2);
          double2 b = ldg128_stream(V + (size_t)pos * kSecPanel, pol_first);
          b.x *= a.cK;
          b.y *= a.cK;
          stg128_stream(Bout + (size_t)m0.x * kSecPanel, b, pol_first);
          sts128(sB + (m0.z >> 16) * 64u + 16u * q, b);
        }
        __syncthreads();
        ++epoch;
        continue;
      }
      const bool p2 = ph == 2;
      if (!p2) {  // row records of the next work item -> L2 (prefetching V as well doubles its DRAM
                  // reads: measured 4.45 GB instead of 2.66 GB per sweep)
        const int4 wn = s_work[(it + 1) & 1];
        if (wn.x < total) {
          l2_prefetch(a.meta + (size_t)wn.y * 2, (unsigned)wn.z * 32u, tid, 0);
        }
      }
      // Row passes work in batches of kBatch x 8 rows per warp (rows dealt out statically: batch t
      // of warp w starts at row (t * warps + w) * 32): all row records of a batch are requested
      // at once, then all global operands, then the rows are finished.  Few load generations
      // with many loads each suit the six scoreboards of a warp; the records of the warp's rows
      // are asked into L1 before the structured passes, which hide that latency.
      constexpr int kBatchRows = kBatch * kTailRows;
      if (p2) {
        mbar_wait(&bar, parity);
        parity ^= 1u;
      }
      structured_v1<G1, NNN, JW>(a, k, units1, &s_ctr[p2 ? 0 : 3], (p2 ? sA : sB) + 8u * l8,
                                 (p2 ? sB : sA) + 8u * l8, p2 ? a.pf : a.ps, p2 ? 0.0 : a.qs,
                                 p2 ? 1.0 : a.rs, p2 || MODE != MODE_INIT, epoch, lane);
      structured_v2<G2, NNN, JW>(a, k, units2, &s_ctr[p2 ? 1 : 4], (p2 ? sA : sB) + 8u * l8,
                                 (p2 ? sB : sA) + 8u * l8, p2 ? a.pf : a.ps, epoch, lane);
      // two register sets in turn (A, B): the records of the next batch are requested before the
      // rows of the current one are finished
      if (p2) {
        auto load_m = [&](RowMeta (&m)[kBatch], int base) {
#pragma unroll
          for (int u = 0; u < kBatch; ++u) m[u] = load_meta(meta, base + slot + u * kTailRows, nrows, true);
        };
        auto load_o = [&](RowOperands (&o)[kBatch], const RowMeta (&m)[kBatch]) {
#pragma unroll
          for (int u = 0; u < kBatch; ++u) o[u] = load_operands(m[u], X1);
        };
        auto finish = [&](int base, const RowMeta (&m)[kBatch], const RowOperands (&o)[kBatch]) {
#pragma unroll
          for (int u = 0; u < kBatch; ++u) {
            const int pos = base + slot + u * kTailRows;
            const uint32_t c0 = m[u].m0.w, c1 = m[u].m1.x, c2 = m[u].m1.y;
            const uint32_t own = (m[u].m0.z >> 16) * 64u + 16u * q;
            double2 y = make_double2(0.0, 0.0);
            fma2(__hiloint2double((int)m[u].m1.w, (int)m[u].m1.z), lds128(sA + own, epoch), y);
            cross_group(m[u], sA + 16u * q, a.t1, a.t2, epoch, y);
            fma2(signed_coef(a.ccoef[(c0 >> kCrossPosBits) & 15u], c0), o[u].h0, y);
            fma2(signed_coef(a.ccoef[(c1 >> kCrossPosBits) & 15u], c1), o[u].h1, y);
            fma2(signed_coef(a.ccoef[(c2 >> kCrossPosBits) & 15u], c2), o[u].h2, y);
            double2 b = lds128(sB + own, epoch);  // P_k + pf O_l b_{k+1}
            b.x = fma(a.pf, y.x, b.x);
            b.y = fma(a.pf, y.y, b.y);
            if (pos < nrows) {
              if (MODE == MODE_LAST) {
                const int dst = __ldg(a.dst_nat + row0 + pos);
                stg128_stream(a.W + (size_t)dst * a.w_ld + panel * kSecPanel + 2 * q, b, pol_first);
              } else {
                stg128_stream(Bout + (size_t)m[u].m0.x * kSecPanel, b, pol_first);
                sts128(sB + own, b);
              }
            }
          }
        };
        RowMeta mA[kBatch], mB[kBatch];
        RowOperands oA[kBatch], oB[kBatch];
        int baseA = claim(&s_ctr[2], kBatchRows, lane), baseB;
        load_m(mA, baseA);
        for (;;) {
          if (baseA >= nrows) break;
          baseB = claim(&s_ctr[2], kBatchRows, lane);
          load_o(oA, mA);
          load_m(mB, baseB);
          finish(baseA, mA, oA);
          if (baseB >= nrows) break;
          baseA = claim(&s_ctr[2], kBatchRows, lane);
          load_o(oB, mB);
          load_m(mA, baseA);
          finish(baseB, mB, oB);
        }
      } else {
        const bool use_v = a.cs != 0.0;
        auto load_mv = [&](RowMeta (&m)[kBatch], double2 (&v)[kBatch], int base) {
#pragma unroll
          for (int u = 0; u < kBatch; ++u) {
            m[u] = load_meta(meta, base + slot + u * kTailRows, nrows, false);
            v[u] = load_stream_if(V, base + slot + u * kTailRows, nrows, use_v, pol_first);
          }
        };
        auto finish = [&](int base, const RowMeta (&m)[kBatch], const double2 (&v)[kBatch]) {
#pragma unroll
          for (int u = 0; u < kBatch; ++u) {
            const int pos = base + slot + u * kTailRows;
            const uint32_t own = (m[u].m0.z >> 16) * 64u + 16u * q;
            double2 z = lds128(sA + own, epoch), g = make_double2(0.0, 0.0);
            cross_group(m[u], sB + 16u * q, a.t1, a.t2, epoch, g);
            z.x = fma(a.cs, v[u].x, fma(a.ps, g.x, z.x));
            z.y = fma(a.cs, v[u].y, fma(a.ps, g.y, z.y));
            if (pos < nrows) stg128_stream(Pout + (size_t)m[u].m0.x * kSecPanel, z, pol_first);
          }
        };
        RowMeta mA[kBatch], mB[kBatch];
        double2 vA[kBatch], vB[kBatch];
        int baseA = claim(&s_ctr[5], kBatchRows, lane), baseB;
        load_mv(mA, vA, baseA);
        for (;;) {
          if (baseA >= nrows) break;
          baseB = claim(&s_ctr[5], kBatchRows, lane);
          load_mv(mB, vB, baseB);
          finish(baseA, mA, vA);
          if (baseB >= nrows) break;
          baseA = claim(&s_ctr[5], kBatchRows, lane);
          load_mv(mA, vA, baseA);
          finish(baseB, mB, vB);
        }
      }
      __syncthreads();  // after phase 3: both buffers are free for the next tile
      ++epoch;
    }
  }
}

// Launch and occupancy entry points of one instantiation file.
template <int M, bool NNN, bool JW>
int launch_sector(const SecArgs& a, int mode, int grid, size_t smem, cudaStream_t st) {
  if (mode == MODE_INIT)
    sector_sweep_kernel<M, NNN, JW, MODE_INIT><<<grid, kSecThreads, smem, st>>>(a);
  else if (mode == MODE_LAST)
    sector_sweep_kernel<M, NNN, JW, MODE_LAST><<<grid, kSecThreads, smem, st>>>(a);
  else
    sector_sweep_kernel<M, NNN, JW, MODE_STEP><<<grid, kSecThreads, smem, st>>>(a);
  POLFED_LAUNCH_CHECK("sector_sweep_kernel");
  return POLFED_OK;
}

template <int M, bool NNN, bool JW, int MODE>
int configure_sector_one(size_t smem, int* occ) {
  POLFED_CUDA(cudaFuncSetAttribute(sector_sweep_kernel<M, NNN, JW, MODE>,
                                   cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int o = 0;
  POLFED_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(
      &o, sector_sweep_kernel<M, NNN, JW, MODE>, kSecThreads, smem));
  if (o < 1) return fail(POLFED_ECUDA, "sector sweep: kernel does not fit an SM");
  *occ = (*occ == 0 || o < *occ) ? o : *occ;
  return POLFED_OK;
}

template <int M, bool NNN, bool JW>
int configure_sector(size_t smem, int* occ) {
  int rc;
  if ((rc = configure_sector_one<M, NNN, JW, MODE_STEP>(smem, occ))) return rc;
  if ((rc = configure_sector_one<M, NNN, JW, MODE_INIT>(smem, occ))) return rc;
  return configure_sector_one<M, NNN, JW, MODE_LAST>(smem, occ);
}

}  // namespace sector
}  // namespace polfed

// Defines the two entry points of one instantiation (declared in sector_sweep.cu).
#define POLFED_SECTOR_DEF(M, NNN, JW)                                                            \
  namespace polfed {                                                                             \
  int sector_launch_##M##_##NNN##_##JW(const sector::SecArgs& a, int mode, int grid, size_t smem, \
                                       cudaStream_t st) {                                        \
    return sector::launch_sector<M, NNN != 0, JW != 0>(a, mode, grid, smem, st);                 \
  }                                                                                              \
  int sector_configure_##M##_##NNN##_##JW(size_t smem, int* occ) {                               \
    return sector::configure_sector<M, NNN != 0, JW != 0>(smem, occ);                            \
  }                                                                                              \
  }
