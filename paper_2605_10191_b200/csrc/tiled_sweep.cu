// The tiled hot path (tiled.cuh): one persistent kernel per Clenshaw step.  A CTA takes a tile
// (a contiguous run of positions that share their high bits), pulls its 16-column panel of
// b_{k+1} into shared memory with one bulk copy, finishes b_k from shared-memory gathers, parks
// b_k in an L2-resident scratch, pulls it back as the new shared tile and starts P_{k-1} from it.
// Eq. (51) PAPER.md:427-431 with the rescaling of Eq. (31); see tiled.cuh for the algebra.
//
// Thread mapping.  Four lanes own one 128-byte panel row, 32 contiguous bytes each, so every
// global access of a row is one 256-bit instruction per lane and one full line per row.  In
// shared memory the same 32 bytes are read as two 16-byte chunks; the rows a warp works on
// alternate the order of the two (even row slots low chunk first, odd slots high chunk first),
// so that the two rows of a quarter-warp always hit disjoint banks whatever rows they gather.
#include <cstdlib>
#include <type_traits>

#include "sector.cuh"
#include "tiled.cuh"

namespace polfed {
namespace {

enum { MODE_STEP = 0, MODE_INIT = 1, MODE_LAST = 2 };

constexpr int kRowsPerIter = 8;  // rows per warp iteration

struct SweepArgs {
  long long n;
  int n_tiles, n_panels, max_tile_rows;
  const int32_t* tile_row0;
  const int32_t* tile_rec0;
  const uint32_t* records;  // kTileRecWords words per class row, position order
  const double* diag;       // [n]
  const uint32_t* side;     // [n][side_words]: other-layout position, packed cross-cut words
  int side_words;
  double ccoef[kTileMaxCrossCoef + 1];
  const int32_t* dst_map;   // position -> output row (other layout, or natural for MODE_LAST)
  double coef[kTileMaxCoef];
  const double* X1;  // b_{k+1}, panel-major, this layout
  const double* Pk;  // partial b_k
  const double* V;   // V in this layout
  double* Bout;      // b_k, other layout
  double* Pout;      // partial b_{k-1}, other layout
  double* W;         // MODE_LAST: row-major n x w_ld output in the caller's row order
  int w_ld;
  double* scratch;   // per CTA: max_tile_rows x 16 doubles
  int* counter;
  double cK;              // MODE_INIT: b_K = cK V
  double pf;              // finishing scalar p_k
  double ps, qs, rs, cs;  // starting scalars of step k-1
  int mode;
};

struct D4 {
  double x, y, z, w;  // x,y = low 16-byte chunk, z,w = high chunk of a lane's 32 bytes
};

__device__ __forceinline__ D4 ldg256(const double* p) {  // read-only data, default caching
  D4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w)
               : "l"(p));
  return r;
}
// L2 policies: block passes that are touched once per sweep leave L2 first, the per-CTA scratch
// and the tile of b_{k+1} (read again by phase 3 and by the neighbours' cross-cut hops) last.
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ D4 ldg256_stream(const double* p, uint64_t pol) {  // touched once
  D4 r;
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f64 {%0,%1,%2,%3}, [%4], %5;"
               : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w)
               : "l"(p), "l"(pol));
  return r;
}
__device__ __forceinline__ void stg256_hint(double* p, const D4& r, uint64_t pol) {
  asm volatile("st.global.L1::no_allocate.L2::cache_hint.v4.f64 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p),
               "d"(r.x), "d"(r.y), "d"(r.z), "d"(r.w), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void stg256(double* p, const D4& r) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(r.x), "d"(r.y), "d"(r.z),
               "d"(r.w)
               : "memory");
}
__device__ __forceinline__ D4 ldg256_plain_stream(const double* p) {
  D4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w)
               : "l"(p));
  return r;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
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
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar,
                                         uint64_t pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], "
      "%2, [%3], %4;" ::"r"(smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async;" ::: "memory");
}

// One thread: bulk-copy `bytes` (a multiple of 128) from global to shared in <= 32 KB pieces.
__device__ __forceinline__ void tile_load(void* dst, const void* src, unsigned bytes, uint64_t* bar,
                                          uint64_t pol) {
  mbar_expect_tx(bar, bytes);
  for (unsigned at = 0; at < bytes; at += 32768u) {
    const unsigned len = min(32768u, bytes - at);
    bulk_g2s(static_cast<char*>(dst) + at, static_cast<const char*>(src) + at, len, bar, pol);
  }
}

template <int NC>
__device__ __forceinline__ double pick_coef(uint32_t cls, const double (&coef)[kTileMaxCoef]) {
  double cf = coef[0];
  if (NC == 2) {
    if (cls & 1u) cf = coef[1];
  } else if (NC > 2) {
    if (cls == 1u) cf = coef[1];
    if (cls == 2u) cf = coef[2];
    if (cls == 3u) cf = coef[3];
  }
  return cf;
}

__device__ __forceinline__ double signed_coef(double cf, uint32_t sign_bit31) {
  return __hiloint2double(__double2hiint(cf) ^ (int)(sign_bit31 & 0x80000000u), __double2loint(cf));
}

// One neighbour: position (x 128 bytes) `off`, amplitude class `cls`, sign in bit 31 of `sg`.
template <int NC>
__device__ __forceinline__ void hop_fma(uint32_t cls, uint32_t sg, uint32_t off,
                                        const unsigned char* __restrict__ x_first,
                                        const unsigned char* __restrict__ x_second,
                                        const double (&coef)[kTileMaxCoef], double2& acc_f,
                                        double2& acc_s) {
  const double cf = signed_coef(pick_coef<NC>(cls, coef), sg);
  const double2 xa = *reinterpret_cast<const double2*>(x_first + off);
  const double2 xb = *reinterpret_cast<const double2*>(x_second + off);
  acc_f.x = fma(cf, xa.x, acc_f.x);
  acc_f.y = fma(cf, xa.y, acc_f.y);
  acc_s.x = fma(cf, xb.x, acc_s.x);
  acc_s.y = fma(cf, xb.y, acc_s.y);
}

// One record word = two neighbours: the quad shuffle of the word and its four 16-byte gathers.
struct HopWord {
  uint32_t word;
  double2 a0, a1, b0, b1;  // neighbour A (first, second chunk), neighbour B
};

__device__ __forceinline__ HopWord hop_fetch(const uint4 rq, int w,
                                             const unsigned char* __restrict__ x_first,
                                             const unsigned char* __restrict__ x_second) {
  const uint32_t mine = (w & 3) == 0 ? rq.x : (w & 3) == 1 ? rq.y : (w & 3) == 2 ? rq.z : rq.w;
  HopWord h;
  h.word = __shfl_sync(0xffffffffu, mine, w >> 2, 4);
  const uint32_t oa = h.word & 0x3ff80u, ob = (h.word >> 11) & 0x3ff80u;
  h.a0 = *reinterpret_cast<const double2*>(x_first + oa);
  h.a1 = *reinterpret_cast<const double2*>(x_second + oa);
  h.b0 = *reinterpret_cast<const double2*>(x_first + ob);
  h.b1 = *reinterpret_cast<const double2*>(x_second + ob);
  return h;
}

template <int NC>
__device__ __forceinline__ void hop_apply(const HopWord& h, const double (&coef)[kTileMaxCoef],
                                          double2& acc_f, double2& acc_s) {
  const double ca = signed_coef(pick_coef<NC>(h.word & 3u, coef), h.word << 1);
  const double cb = signed_coef(pick_coef<NC>((h.word >> 2) & 3u, coef), h.word);
  acc_f.x = fma(ca, h.a0.x, acc_f.x);
  acc_f.y = fma(ca, h.a0.y, acc_f.y);
  acc_s.x = fma(ca, h.a1.x, acc_s.x);
  acc_s.y = fma(ca, h.a1.y, acc_s.y);
  acc_f.x = fma(cb, h.b0.x, acc_f.x);
  acc_f.y = fma(cb, h.b0.y, acc_f.y);
  acc_s.x = fma(cb, h.b1.x, acc_s.x);
  acc_s.y = fma(cb, h.b1.y, acc_s.y);
}

// All in-tile neighbours of the row whose record quarter this lane holds (rq); max_deg is
// warp-uniform, shorter rows run into entries that point at the zero row.  The gathers of word
// w + 1 are issued before the FMAs of word w.
template <int NC>
__device__ __forceinline__ void tile_hops(const uint4 rq, int max_deg,
                                          const unsigned char* __restrict__ x_first,
                                          const unsigned char* __restrict__ x_second,
                                          const double (&coef)[kTileMaxCoef], double2& acc_f,
                                          double2& acc_s) {
  if (max_deg <= 0) return;
  HopWord cur = hop_fetch(rq, 1, x_first, x_second);
#pragma unroll
  for (int w = 1; w <= kTileMaxDeg / 2; ++w) {
    HopWord nxt = cur;
    const bool more = w < kTileMaxDeg / 2 && 2 * w < max_deg;
    if (more) nxt = hop_fetch(rq, w + 1, x_first, x_second);
    hop_apply<NC>(cur, coef, acc_f, acc_s);
    if (!more) break;
    cur = nxt;
  }
}

// (first, second) accumulators of a lane -> (low, high) chunk order of its 32 bytes.
__device__ __forceinline__ D4 to_lohi(const double2 f, const double2 s, bool odd) {
  D4 r;
  r.x = odd ? s.x : f.x;
  r.y = odd ? s.y : f.y;
  r.z = odd ? f.x : s.x;
  r.w = odd ? f.y : s.y;
  return r;
}

__device__ __forceinline__ void d4_zero(D4& r) { r.x = r.y = r.z = r.w = 0.0; }
__device__ __forceinline__ void d4_fma(double c, const D4& g, D4& acc) {
  acc.x = fma(c, g.x, acc.x);
  acc.y = fma(c, g.y, acc.y);
  acc.z = fma(c, g.z, acc.z);
  acc.w = fma(c, g.w, acc.w);
}

constexpr uint32_t kCrossPosMask = (1u << kCrossPosBits) - 1u;

// What phase 2 needs of a row before its tile hops: the record quarter, the side record
// (position in the other layout + first three cross-cut words) and the diagonal.  Loaded one
// iteration ahead, so that the cross-cut gathers can be issued before the hops.
struct RowHead {
  uint4 rq;
  uint4 side;
  double dg;
};

__device__ __forceinline__ RowHead load_head(const uint4* rec, const uint32_t* side_row0,
                                             int side_words, const double* diag_row0, int pos,
                                             int nrows, int q) {
  RowHead h;
  h.rq = make_uint4(0u, 0u, 0u, 0u);
  h.side = make_uint4(0u, kCrossNone, kCrossNone, kCrossNone);
  h.dg = 0.0;
  if (pos < nrows) {
    h.rq = __ldg(rec + (size_t)pos * 4 + q);
    h.side = __ldg(reinterpret_cast<const uint4*>(side_row0 + (size_t)pos * side_words));
    h.dg = __ldg(diag_row0 + pos);
  }
  return h;
}

// A warp claims the next kRowsPerIter positions of the tile (rows are sorted by falling degree,
// so claiming in order also balances the warps).
__device__ __forceinline__ int grab_chunk(int* counter, int lane) {
  int v = 0;
  if (lane == 0) v = atomicAdd(counter, kRowsPerIter);
  return __shfl_sync(0xffffffffu, v, 0);
}

// THREADS = 512 with one CTA per SM for tiles that fill the shared memory, 256 with three CTAs
// per SM (85 registers) for tiles of at most a third of it.
// Same for a work item = (panel, tile) of the panel-major order of the row-record sweep.
__device__ __forceinline__ void next_work_prefetch(const SweepArgs& a, int work_n,
                                                   size_t panel_stride, int tid) {
  if (work_n >= a.n_tiles * a.n_panels) return;
  const int tile = work_n % a.n_tiles, npanel = work_n / a.n_tiles;
  const int row0 = __ldg(a.tile_row0 + tile);
  const unsigned bytes = (unsigned)(__ldg(a.tile_row0 + tile + 1) - row0) * 128u;
  const unsigned at = (unsigned)tid * 2048u;
  if (at < bytes)
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(
                     a.X1 + npanel * panel_stride + (size_t)row0 * kTilePanel + at / 8),
                 "r"(min(2048u, bytes - at))
                 : "memory");
}

// Register cap instead of launch bounds: 152 lets ptxas settle on 110 registers for the 384-thread
// variant (4.62 ms per sweep on config 5; __launch_bounds__(384, 1): 115 registers, 4.69 ms;
// cap 128: 4.67; cap 104: 5.5).
template <int NC, int MODE, int THREADS>
__global__ void __maxnreg__(THREADS == kTileThreads ? 152 : 80)
    tiled_sweep_kernel(const SweepArgs a) {
  constexpr int kIterRows = (THREADS / 32) * kRowsPerIter;  // rows per CTA pass (static loops)
  extern __shared__ __align__(128) unsigned char smem_raw[];  // (max_tile_rows + 1) x 128 B
  __shared__ uint64_t bar;
  __shared__ int4 s_tile[2];  // work item, first row, rows, first record of the tile's class
  __shared__ int s_chunk[2];  // next unclaimed position of the running phase / the one after it
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int q = lane & 3, slot = lane >> 2;
  const bool odd = slot & 1;
  const unsigned char* x_first = smem_raw + 32 * q + (odd ? 16 : 0);
  const unsigned char* x_second = smem_raw + 32 * q + (odd ? 0 : 16);
  const int total = a.n_tiles * a.n_panels;
  auto next_work = [&]() {  // one thread: claim a work item and look its tile up
    int4 w = make_int4(atomicAdd(a.counter, 1), 0, 0, 0);
    if (w.x < total) {
      const int tile = w.x % a.n_tiles;
      w.y = __ldg(a.tile_row0 + tile);
      w.z = __ldg(a.tile_row0 + tile + 1) - w.y;
      w.w = __ldg(a.tile_rec0 + tile);
    }
    return w;
  };
  if (tid == 0) {
    mbar_init(&bar, 1);
    s_tile[0] = next_work();
    s_chunk[0] = s_chunk[1] = 0;
  }
  __syncthreads();
  unsigned parity = 0;
  int phase = 0;  // selects the chunk counter; the other one is reset at the start of a phase
  double* scratch = a.scratch + (size_t)blockIdx.x * a.max_tile_rows * kTilePanel;
  const size_t panel_stride = (size_t)a.n * kTilePanel;  // doubles per panel
  const double2 zero2 = make_double2(0.0, 0.0);
  const int first_pos = warp * kRowsPerIter + slot;
  const uint64_t pol_first = l2_policy_evict_first(), pol_last = l2_policy_evict_last();

  for (int it = 0;; ++it) {
    // work items in panel-major order: all tiles of panel 0, then panel 1 (half the live X in L2)
    const int4 wi = s_tile[it & 1];
    const int work = wi.x, row0 = wi.y, nrows = wi.z;
    if (work >= total) break;
    const int panel_of_work = work / a.n_tiles;
    const uint4* rec = reinterpret_cast<const uint4*>(a.records) + (size_t)wi.w * 4;
    const uint32_t* side = a.side + (size_t)row0 * a.side_words;
    const double* diag = a.diag + row0;
    const int32_t* dst_map = a.dst_map + row0;
    if (tid < 8) reinterpret_cast<double2*>(smem_raw)[nrows * 8 + tid] = zero2;  // the zero row
    __syncthreads();
    // the next work item is claimed by the last warp (only its lane 0 waits for the atomic and the
    // tile look-up) and read after later barriers
    if (tid == THREADS - 32) s_tile[(it + 1) & 1] = next_work();

    for (int panel = panel_of_work; panel == panel_of_work; ++panel) {
      const double* X1 = a.X1 + panel * panel_stride;
      const double* Pk = a.Pk + panel * panel_stride + (size_t)row0 * kTilePanel;
      const double* V = a.V + panel * panel_stride + (size_t)row0 * kTilePanel;
      double* Bout = a.Bout + panel * panel_stride;
      double* Pout = a.Pout + panel * panel_stride;

      if (MODE == MODE_INIT) {
        // ---- b_K = c_K V ------------------------------------------------------------------------
        for (int pos = first_pos; pos < nrows; pos += kIterRows) {
          const int dst = __ldg(dst_map + pos);
          D4 b = ldg256_stream(V + (size_t)pos * kTilePanel + 4 * q, pol_first);
          b.x *= a.cK;
          b.y *= a.cK;
          b.z *= a.cK;
          b.w *= a.cK;
          stg256_hint(Bout + (size_t)dst * kTilePanel + 4 * q, b, pol_first);
          stg256_hint(scratch + (size_t)pos * kTilePanel + 4 * q, b, pol_last);
        }
      } else {
        // ---- phase 2: b_k = P_k + p_k (O_l + DM) b_{k+1} ---------------------------------------
        if (tid == 0)
          tile_load(smem_raw, X1 + (size_t)row0 * kTilePanel, (unsigned)nrows * 128u, &bar,
                    pol_last);
        if (tid == 0) s_chunk[(phase + 1) & 1] = 0;
        int* const chunk = &s_chunk[phase & 1];
        ++phase;
        int base = grab_chunk(chunk, lane), base_n = grab_chunk(chunk, lane);
        RowHead nx = load_head(rec, side, a.side_words, diag, base + slot, nrows, q);
        mbar_wait(&bar, parity);
        parity ^= 1u;
        for (; base < nrows; base = base_n, base_n = grab_chunk(chunk, lane)) {
          const int pos = base + slot;
          const bool active = pos < nrows;
          const RowHead hd = nx;
          nx = load_head(rec, side, a.side_words, diag, base_n + slot, nrows, q);
          // this row's stream and the cross-cut rows (other tiles, from L2) fly during the hops
          D4 pk, g0, g1, g2;
          d4_zero(pk);
          d4_zero(g0);
          d4_zero(g1);
          d4_zero(g2);
          int dst = (int)hd.side.x;
          if (active) {
            pk = ldg256_stream(Pk + (size_t)pos * kTilePanel + 4 * q, pol_first);
            if (MODE == MODE_LAST) dst = __ldg(dst_map + pos);
          }
          if (hd.side.y != kCrossNone)
            g0 = ldg256(X1 + (size_t)(hd.side.y & kCrossPosMask) * kTilePanel + 4 * q);
          if (hd.side.z != kCrossNone)
            g1 = ldg256(X1 + (size_t)(hd.side.z & kCrossPosMask) * kTilePanel + 4 * q);
          if (hd.side.w != kCrossNone)
            g2 = ldg256(X1 + (size_t)(hd.side.w & kCrossPosMask) * kTilePanel + 4 * q);
          const int deg = __shfl_sync(0xffffffffu, (int)hd.rq.x, 0, 4);
          const int max_deg = __reduce_max_sync(0xffffffffu, deg);
          double2 acc_f = zero2, acc_s = zero2;
          tile_hops<NC>(hd.rq, max_deg, x_first, x_second, a.coef, acc_f, acc_s);
          if (active) {  // diagonal: own row of the shared tile
            const double2 oa = *reinterpret_cast<const double2*>(x_first + (size_t)pos * 128);
            const double2 ob = *reinterpret_cast<const double2*>(x_second + (size_t)pos * 128);
            acc_f.x = fma(hd.dg, oa.x, acc_f.x);
            acc_f.y = fma(hd.dg, oa.y, acc_f.y);
            acc_s.x = fma(hd.dg, ob.x, acc_s.x);
            acc_s.y = fma(hd.dg, ob.y, acc_s.y);
          }
          D4 acc = to_lohi(acc_f, acc_s, odd);
          d4_fma(signed_coef(a.ccoef[(hd.side.y >> kCrossPosBits) & 15u], hd.side.y), g0, acc);
          d4_fma(signed_coef(a.ccoef[(hd.side.z >> kCrossPosBits) & 15u], hd.side.z), g1, acc);
          d4_fma(signed_coef(a.ccoef[(hd.side.w >> kCrossPosBits) & 15u], hd.side.w), g2, acc);
          if (a.side_words > 4 && active) {  // cross-cut words 3..6 (wide cuts only)
            const uint4 more = __ldg(reinterpret_cast<const uint4*>(side + (size_t)pos * 8 + 4));
            const uint32_t cw[4] = {more.x, more.y, more.z, more.w};
#pragma unroll
            for (int j = 0; j < 4; ++j)
              if (cw[j] != kCrossNone) {
                const D4 g = ldg256(X1 + (size_t)(cw[j] & kCrossPosMask) * kTilePanel + 4 * q);
                d4_fma(signed_coef(a.ccoef[(cw[j] >> kCrossPosBits) & 15u], cw[j]), g, acc);
              }
          }
          D4 b;
          b.x = fma(a.pf, acc.x, pk.x);
          b.y = fma(a.pf, acc.y, pk.y);
          b.z = fma(a.pf, acc.z, pk.z);
          b.w = fma(a.pf, acc.w, pk.w);
          if (active) {
            if (MODE == MODE_LAST) {
              stg256_hint(a.W + (size_t)dst * a.w_ld + panel * kTilePanel + 4 * q, b, pol_first);
            } else {
              stg256_hint(Bout + (size_t)dst * kTilePanel + 4 * q, b, pol_first);
              stg256_hint(scratch + (size_t)pos * kTilePanel + 4 * q, b, pol_last);
            }
          }
        }
      }
      if (MODE == MODE_LAST) {
        __syncthreads();  // the next bulk copy overwrites the tile
        continue;
      }

      // ---- b_k becomes the shared tile ------------------------------------------------------
      __threadfence_block();
      fence_proxy_async();
      __syncthreads();
      if (tid == 0) {
        tile_load(smem_raw, scratch, (unsigned)nrows * 128u, &bar, pol_last);
        s_chunk[(phase + 1) & 1] = 0;
      }
      int* const chunk = &s_chunk[phase & 1];
      ++phase;
      int base = grab_chunk(chunk, lane), base_n = grab_chunk(chunk, lane);
      uint4 rq_n = make_uint4(0u, 0u, 0u, 0u);
      if (base + slot < nrows) rq_n = __ldg(rec + (size_t)(base + slot) * 4 + q);
      if (MODE == MODE_STEP)
        next_work_prefetch(a, s_tile[(it + 1) & 1].x, panel_stride, tid);
      mbar_wait(&bar, parity);
      parity ^= 1u;
      // the parked copy is dead once it is back in shared memory: drop it from L2 unwritten
      for (int r = tid; r < nrows; r += THREADS)
        asm volatile("discard.global.L2 [%0], 128;" ::"l"(scratch + (size_t)r * kTilePanel) : "memory");

      // ---- phase 3: P_{k-1} = c_{k-1} V + p_{k-1} O_l b_k + q_{k-1} b_k + r b_{k+1} ------------
      for (; base < nrows; base = base_n, base_n = grab_chunk(chunk, lane)) {
        const int pos = base + slot;
        const bool active = pos < nrows;
        const uint4 rq = rq_n;
        {
          const int pos_n = base_n + slot;
          rq_n = make_uint4(0u, 0u, 0u, 0u);
          if (pos_n < nrows) rq_n = __ldg(rec + (size_t)pos_n * 4 + q);
        }
        D4 x1, v;
        d4_zero(x1);
        d4_zero(v);
        int dst = 0;
        if (active) {
          dst = __ldg(dst_map + pos);
          if (a.rs != 0.0) x1 = ldg256(X1 + ((size_t)row0 + pos) * kTilePanel + 4 * q);
          if (a.cs != 0.0) v = ldg256_stream(V + (size_t)pos * kTilePanel + 4 * q, pol_first);
        }
        const int deg = __shfl_sync(0xffffffffu, (int)rq.x, 0, 4);
        const int max_deg = __reduce_max_sync(0xffffffffu, deg);
        double2 acc_f = zero2, acc_s = zero2;
        tile_hops<NC>(rq, max_deg, x_first, x_second, a.coef, acc_f, acc_s);
        if (active) {
          const double2 oa = *reinterpret_cast<const double2*>(x_first + (size_t)pos * 128);
          const double2 ob = *reinterpret_cast<const double2*>(x_second + (size_t)pos * 128);
          acc_f.x = fma(a.ps, acc_f.x, a.qs * oa.x);
          acc_f.y = fma(a.ps, acc_f.y, a.qs * oa.y);
          acc_s.x = fma(a.ps, acc_s.x, a.qs * ob.x);
          acc_s.y = fma(a.ps, acc_s.y, a.qs * ob.y);
          D4 y = to_lohi(acc_f, acc_s, odd);
          y.x = fma(a.cs, v.x, fma(a.rs, x1.x, y.x));
          y.y = fma(a.cs, v.y, fma(a.rs, x1.y, y.y));
          y.z = fma(a.cs, v.z, fma(a.rs, x1.z, y.z));
          y.w = fma(a.cs, v.w, fma(a.rs, x1.w, y.w));
          stg256_hint(Pout + (size_t)dst * kTilePanel + 4 * q, y, pol_first);
        }
      }
      __syncthreads();  // all reads of the tile done before the next bulk copy
    }
  }
}

// V (row-major n x s, caller's row order) -> panel-major copies at the positions of both layouts.
__global__ void __launch_bounds__(256) tiled_pack_kernel(long long n, int n_panels,
                                                         const double* __restrict__ V,
                                                         const int32_t* __restrict__ from_nat0,
                                                         const int32_t* __restrict__ from_nat1,
                                                         double* __restrict__ V0,
                                                         double* __restrict__ V1) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;  // one 32-byte piece each
  const int per_row = n_panels * 4;
  const long long row = t / per_row;
  if (row >= n) return;
  const int w = (int)(t % per_row), panel = w >> 2, piece = w & 3;
  const D4 v = ldg256_plain_stream(V + t * 4);
  const size_t ps = (size_t)n * kTilePanel;
  stg256(V0 + panel * ps + (size_t)__ldg(from_nat0 + row) * kTilePanel + 4 * piece, v);
  stg256(V1 + panel * ps + (size_t)__ldg(from_nat1 + row) * kTilePanel + 4 * piece, v);
}

template <int NC, int THREADS>
int launch_sweep_t(const TiledPlan* p, const SweepArgs& a, cudaStream_t st) {
  if (a.mode == MODE_INIT)
    tiled_sweep_kernel<NC, MODE_INIT, THREADS><<<p->grid, THREADS, p->smem_bytes, st>>>(a);
  else if (a.mode == MODE_LAST)
    tiled_sweep_kernel<NC, MODE_LAST, THREADS><<<p->grid, THREADS, p->smem_bytes, st>>>(a);
  else
    tiled_sweep_kernel<NC, MODE_STEP, THREADS><<<p->grid, THREADS, p->smem_bytes, st>>>(a);
  POLFED_LAUNCH_CHECK("tiled_sweep_kernel");
  return POLFED_OK;
}

template <int NC>
int launch_sweep(const TiledPlan* p, const SweepArgs& a, cudaStream_t st) {
  return p->threads == kTileThreads ? launch_sweep_t<NC, kTileThreads>(p, a, st)
                                    : launch_sweep_t<NC, kTileSmallThreads>(p, a, st);
}

int sweep(const TiledPlan* p, int layout, SweepArgs a, cudaStream_t st) {
  const TiledLayout& L = p->lay[layout];
  a.records = L.d_records;
  a.diag = L.d_diag;
  a.side = L.d_side;
  a.side_words = L.side_words;
  for (int c = 0; c <= kTileMaxCrossCoef; ++c) a.ccoef[c] = L.ccoef[c];
  a.dst_map = (a.mode == MODE_LAST) ? L.d_to_natural : L.d_to_other;
  for (int c = 0; c < kTileMaxCoef; ++c) a.coef[c] = L.coef[c];
  POLFED_CUDA(cudaMemsetAsync(a.counter, 0, sizeof(int), st));
  return L.n_coef <= 2 ? launch_sweep<2>(p, a, st) : launch_sweep<4>(p, a, st);
}

template <int NC, int MODE, int THREADS>
int configure_one(TiledPlan* p, int* occ) {
  POLFED_CUDA(cudaFuncSetAttribute(tiled_sweep_kernel<NC, MODE, THREADS>,
                                   cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)p->smem_bytes));
  int o = 0;
  POLFED_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(
      &o, tiled_sweep_kernel<NC, MODE, THREADS>, THREADS, p->smem_bytes));
  if (o < 1) return fail(POLFED_ECUDA, "tiled format: sweep kernel does not fit an SM");
  *occ = (*occ == 0 || o < *occ) ? o : *occ;
  return POLFED_OK;
}

template <int THREADS>
int configure_all(TiledPlan* p, int* occ) {
  int rc;
  if ((rc = configure_one<2, MODE_STEP, THREADS>(p, occ))) return rc;
  if ((rc = configure_one<2, MODE_INIT, THREADS>(p, occ))) return rc;
  if ((rc = configure_one<2, MODE_LAST, THREADS>(p, occ))) return rc;
  if ((rc = configure_one<4, MODE_STEP, THREADS>(p, occ))) return rc;
  if ((rc = configure_one<4, MODE_INIT, THREADS>(p, occ))) return rc;
  if ((rc = configure_one<4, MODE_LAST, THREADS>(p, occ))) return rc;
  return POLFED_OK;
}

}  // namespace

int tiled_configure_launch(TiledPlan* p) {
  p->smem_bytes = (size_t)(p->max_tile_rows + 1) * 128;  // + the zero row
  int occ = 0, rc;
  // small tiles: several CTAs per SM hide each other's bulk-copy waits and barriers
  p->threads = (p->smem_bytes + 1024) * kTileSmallCtas <= 227u * 1024u ? kTileSmallThreads
                                                                        : kTileThreads;
  if (p->threads == kTileThreads) {
    if ((rc = configure_all<kTileThreads>(p, &occ))) return rc;
  } else {
    if ((rc = configure_all<kTileSmallThreads>(p, &occ))) return rc;
  }
  int dev = 0, sms = 148;
  POLFED_CUDA(cudaGetDevice(&dev));
  POLFED_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const long long want = (long long)occ * sms;
  p->grid = (int)(want < p->n_tiles ? want : p->n_tiles);
  if (p->grid < 1) p->grid = 1;
  return POLFED_OK;
}

bool tiled_supports(const polfed_ham* ham, int s) {
  return ham && ham->tiled && (s == 16 || s == 32) && ham->n > 0;
}

size_t sector_workspace_bytes(const polfed_ham* ham, int s);  // sector_sweep.cu
int sector_filter_apply(const polfed_ham* ham, double a, double b, int K, const double* c, int s,
                        const double* d_V, double* d_W, void* d_work, cudaStream_t st);

// X/P pairs (4 blocks) + V in both layouts (2 blocks) + the per-CTA scratch + the tile counter
size_t tiled_workspace_bytes(const polfed_ham* ham, int s) {
  const TiledPlan* p = ham->tiled;
  if (p->sector) return sector_workspace_bytes(ham, s);
  return (size_t)6 * (size_t)ham->n * s * sizeof(double) +
         (size_t)p->grid * p->max_tile_rows * 128 + 128;
}

int tiled_filter_apply(const polfed_ham* ham, double a_, double b_, int K, const double* c,
                       int s, const double* d_V, double* d_W, void* d_work, cudaStream_t st) {
  const TiledPlan* p = ham->tiled;
  if (p->sector) return sector_filter_apply(ham, a_, b_, K, c, s, d_V, d_W, d_work, st);
  const size_t len = (size_t)ham->n * s;
  double* base = static_cast<double*>(d_work);
  double* X[2] = {base, base + 2 * len};
  double* P[2] = {base + len, base + 3 * len};
  double* Vl[2] = {base + 4 * len, base + 5 * len};
  double* scratch = base + 6 * len;
  const int n_panels = s / kTilePanel;

  const long long threads = (long long)ham->n * n_panels * 4;
  tiled_pack_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
      ham->n, n_panels, d_V, p->lay[0].d_from_natural, p->lay[1].d_from_natural, Vl[0], Vl[1]);
  POLFED_LAUNCH_CHECK("tiled_pack_kernel");

  SweepArgs a{};
  a.n = ham->n;
  a.n_tiles = p->n_tiles;
  a.n_panels = n_panels;
  a.max_tile_rows = p->max_tile_rows;
  a.tile_row0 = p->d_tile_row0;
  a.tile_rec0 = p->d_tile_rec0;
  a.scratch = scratch;
  // the tile counter lives in the caller's workspace, so the handle stays read-only
  a.counter = reinterpret_cast<int*>(scratch + (size_t)p->grid * p->max_tile_rows * kTilePanel);
  a.W = d_W;
  a.w_ld = s;
  auto pk = [&](int k) { return (k == 0 ? 1.0 : 2.0) / b_; };
  auto qk = [&](int k) { return (k == 0 ? -1.0 : -2.0) * a_ / b_; };

  // sweep j finishes b_{K-j} in layout j & 1 and starts the partial b_{K-j-1}
  for (int j = 0; j <= K; ++j) {
    const int k = K - j, layout = j & 1;
    const int in = (j + 1) & 1, out = j & 1;  // buffer pairs
    a.X1 = X[in];
    a.Pk = P[in];
    a.V = Vl[layout];
    a.Bout = X[out];
    a.Pout = P[out];
    a.cK = c[K];
    a.pf = pk(k);
    a.mode = (j == 0) ? MODE_INIT : (k == 0 ? MODE_LAST : MODE_STEP);
    if (k > 0) {
      a.ps = pk(k - 1);
      a.qs = qk(k - 1);
      a.cs = c[k - 1];
      a.rs = (j == 0) ? 0.0 : -1.0;
    }
    int rc = sweep(p, layout, a, st);
    if (rc) return rc;
  }
  return POLFED_OK;
}

}  // namespace polfed
