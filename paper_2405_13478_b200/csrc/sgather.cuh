// sgather.cuh -- phase S (gridding, steps a1/a2) as a table-driven gather through
// shared memory, shared by blink_grid (k_grid_ring) and blink_grid_image (k_fused): the device side
// (mbarrier / bulk-copy helpers, the per-warp group loop) and the host side (cells dealt to warps,
// conflict-aware packing of each chunk's gather table).  See blink_fused.cu for the whole picture.
#pragma once

#include <algorithm>
#include <array>
#include <cstring>
#include <vector>

#include "blink_internal.h"
#include "sphase.cuh"

namespace blink {

constexpr int kFusedThreads = 512;
constexpr int kFusedWarps = kFusedThreads / 32;
constexpr int kFusedMaxGroups = 16;   // groups per (warp, chunk): their lengths fit one 32-bit word
constexpr int kFusedLcap = 4;         // rows per group: longer per-chunk cell lists are split into pieces

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!done);
}
// bulk copy global -> shared of `bytes` (multiple of 16, both addresses 16-byte aligned); SASS UBLKCP
__device__ __forceinline__ void bulk_load(void *sdst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(sdst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ uint2 lds_u2(uint32_t addr) {
  uint2 r;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(addr));
  return r;
}

// Phase S works through a warp's groups with a one-group software pipeline: the index column of
// the next group (slot of the cell sum, kFusedLcap entries -- rows beyond the group's L are read
// too and ignored) is requested before the visibilities of the current group are gathered, so a
// group costs about one shared-memory latency instead of three.
struct GroupIdx {
  uint32_t j;
  int e[kFusedLcap];     // sign-extended: conj (bit 15) lands in the sign bit
};

template <int ROWS> __device__ __forceinline__ void load_idx(GroupIdx &gi, uint32_t blk) {
  asm volatile("ld.shared.u16 %0, [%1];" : "=r"(gi.j) : "r"(blk));
#pragma unroll
  for (int r = 0; r < ROWS; ++r) asm volatile("ld.shared.s16 %0, [%1];" : "=r"(gi.e[r]) : "r"(blk + 64u * (r + 1)));
}

// lane l adds its L visibilities and folds the sum into its cell.  CORR: every visibility is first
// multiplied by its pre-gridding correction factor F (blink_correct.cu), which
// arrived in the same buffer f_off bytes behind it -- the corrections "fused at load" of SURVEY 8(f) f2.
template <int L, bool CORR>
__device__ __forceinline__ void fold_group(const GroupIdx &gi, uint32_t sm_base, uint32_t S_base, uint32_t f_base) {
  float2 v[L], a;
#pragma unroll
  for (int r = 0; r < L; ++r) {
    if constexpr (CORR) {
      float2 x, f;
      asm volatile("{\n.reg .b32 t, u;\nand.b32 t, %4, 0x7FFF;\nmad.lo.u32 u, t, 8, %6;\nmad.lo.u32 t, t, 8, %5;\n"
                   "ld.shared.v2.f32 {%0, %1}, [t];\nld.shared.v2.f32 {%2, %3}, [u];\n}"
                   : "=f"(x.x), "=f"(x.y), "=f"(f.x), "=f"(f.y) : "r"(gi.e[r]), "r"(sm_base), "r"(f_base));
      v[r].x = x.x * f.x - x.y * f.y;
      v[r].y = x.x * f.y + x.y * f.x;
    } else {
      asm volatile("{\n.reg .b32 t;\nand.b32 t, %2, 0x7FFF;\nmad.lo.u32 t, t, 8, %3;\nld.shared.v2.f32 {%0, %1}, [t];\n}"
                   : "=f"(v[r].x), "=f"(v[r].y) : "r"(gi.e[r]), "r"(sm_base));
    }
  }
  uint32_t sa;
  asm volatile("mad.lo.u32 %2, %3, 8, %4;\nld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(a.x), "=f"(a.y), "=r"(sa) : "r"(gi.j), "r"(S_base));
#if defined(BLINK_PHASE_S_PACKED)
  // packed fp32 pairs (SASS FADD2): one issue slot per visibility added; same sums in the same order
#pragma unroll
  for (int r = 0; r < L; ++r) v[r].y = __uint_as_float(__float_as_uint(v[r].y) ^ ((uint32_t)gi.e[r] & 0x80000000u));
  unsigned long long acc = reinterpret_cast<const unsigned long long &>(v[0]);
#pragma unroll
  for (int r = 1; r < L; ++r)
    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(acc) : "l"(reinterpret_cast<const unsigned long long &>(v[r])));
  {
    unsigned long long aa = reinterpret_cast<const unsigned long long &>(a);
    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(aa) : "l"(acc));
    a = reinterpret_cast<const float2 &>(aa);
  }
#else
  float ax = v[0].x, ay = __uint_as_float(__float_as_uint(v[0].y) ^ ((uint32_t)gi.e[0] & 0x80000000u));
#pragma unroll
  for (int r = 1; r < L; ++r) {
    ax += v[r].x;
    ay += __uint_as_float(__float_as_uint(v[r].y) ^ ((uint32_t)gi.e[r] & 0x80000000u));
  }
  a.x += ax;
  a.y += ay;
#endif
  asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(sa), "f"(a.x), "f"(a.y) : "memory");
}

// One warp's share of a chunk: `tab` is the shared address of the chunk's gather table (it follows
// the visibilities in the same buffer).  wd.x = offset of the warp's stream | number of groups << 24,
// wd.y = how many of them have L = 4, 3, 2, 1 rows (one byte each, L = 4 in the low byte); the stream
// holds them in that order, so each length class is a tight loop of its own with no per-group dispatch.
template <int L, bool CORR>
__device__ __forceinline__ void consume_class(int n, uint32_t &blk, GroupIdx &ga, GroupIdx &gb, uint32_t sm_base,
                                              uint32_t S_base, uint32_t f_base) {
  // ga holds the index set of the class's first group; on return it holds that of the next class's first
  // group (rows beyond a group's own L are loaded too and ignored; past the last group of the stream the
  // bytes that follow are read, unused)
  while (n >= 2) {
    blk += (L + 1) * 64;
    load_idx<L>(gb, blk);
    fold_group<L, CORR>(ga, sm_base, S_base, f_base);
    blk += (L + 1) * 64;
    load_idx<L>(ga, blk);
    fold_group<L, CORR>(gb, sm_base, S_base, f_base);
    n -= 2;
  }
  if (n) {
    blk += (L + 1) * 64;
    load_idx<L>(gb, blk);
    fold_group<L, CORR>(ga, sm_base, S_base, f_base);
    ga = gb;
  }
}

template <bool CORR = false>
__device__ __forceinline__ void consume_chunk(uint32_t tab, int warp, int lane, uint32_t sm_base, uint32_t S_base,
                                              uint32_t f_off = 0) {
  const uint32_t f_base = sm_base + f_off;   // a visibility in slot s has its factor at f_base + 8 s
  const uint2 wd = lds_u2(tab + 8u * warp);
  uint32_t blk = tab + (wd.x & 0xFFFFFFu) + 2u * lane;
  GroupIdx ga, gb;                         // two index sets, used alternately
  load_idx<kFusedLcap>(ga, blk);
  consume_class<4, CORR>((int)(wd.y & 0xFFu), blk, ga, gb, sm_base, S_base, f_base);
  consume_class<3, CORR>((int)((wd.y >> 8) & 0xFFu), blk, ga, gb, sm_base, S_base, f_base);
  consume_class<2, CORR>((int)((wd.y >> 16) & 0xFFu), blk, ga, gb, sm_base, S_base, f_base);
  consume_class<1, CORR>((int)(wd.y >> 24), blk, ga, gb, sm_base, S_base, f_base);
}

// ---------------------------------------------------------------------------------------------
// Host: phase-S gather tables and the shared-memory plan of the route.
//
// Cells are dealt to the kFusedWarps warps once per channel (longest first, to the least loaded
// warp) and numbered so that the cells of a warp cycle through the 16 shared-memory banks (an
// 8-byte slot's bank is slot mod 16).  For a chunk [lo, hi) of baselines and a warp, each of the
// warp's cells with baselines in the chunk gives one piece (its baselines in the chunk), or several
// pieces of at most kFusedLcap baselines.  The pieces are packed, longest first, into groups of 32
// lanes (two half-warps of 16) of L <= kFusedLcap rows: a piece goes to the lane and rows where it
// collides least with what is already there -- in a half-warp the 16 cell sums should sit in 16
// different banks, and so should the 16 visibilities of every row -- so the shared-memory reads of
// the inner loop are (nearly) conflict-free.  Pieces of one cell never share a group.  Table of one
// (channel, chunk), all offsets in bytes from its start:
//   [0, 128)                per warp: uint32 offset of its stream | number of groups << 24, uint32 with the
//                           number of groups of L = 4, 3, 2, 1 rows (one byte each, L = 4 in the low byte)
//   stream of a warp:       groups in descending L; per group: uint16 j[32]  slot of the cell sum in S
//                             (empty lanes: the zero slot of a bank the half-warp does not use)
//                           L rows of uint16 e[32]: slot | conj << 15, where slot is the visibility's
//                             position in shared memory in 8-byte units (padding: a zero slot in a
//                             bank the half-row does not use)
// L of the gi-th group of a warp's stream, from the class counts of its header word
static inline int group_len(uint32_t counts, int gi) {
  int L = kFusedLcap;
  for (; L > 1; --L, counts >>= 8) {
    if (gi < (int)(counts & 0xFFu)) return L;
    gi -= (int)(counts & 0xFFu);
  }
  return 1;
}

struct AbstractTable {           // entries still relative to the chunk: (bl - lo) | conj << 15, 0x7FFF = padding
  std::vector<unsigned char> bytes;
  long rows = 0, halfrow_wavefronts = 0, groups = 0, rmw_wavefronts = 0;   // statistics
  long warp_cost[16] = {};       // estimated issue slots per warp (see fused_build's rebalancing)
};

constexpr int kGroupCost = 22, kRowCost = 8;   // instructions per group / per row of phase S (from the SASS)

struct FusedPiece { int32_t len, slot, first; };   // first: index into HostGather::src

struct PackGroup {
  int L = 0;
  int n[2] = {0, 0};                       // lanes used per half
  uint32_t sbank[2] = {0, 0};              // banks of the cell sums per half (bit mask)
  int scount[2][16] = {};                  // cell sums per bank per half
  int bcount[2][kFusedLcap][16] = {};      // visibilities per bank per half-row
  std::vector<int32_t> cells;              // slots of the cells in the group
  int32_t lane_slot[32];
  int32_t lane_entry[32][kFusedLcap];      // index into HostGather::src or -1
};

static void build_chunk_table(const HostGather &g, const std::vector<int> &owner, const std::vector<int> &slot,
                              int lo, int hi, int sink0, AbstractTable &out, bool &ok) {
  std::vector<std::vector<FusedPiece>> pieces(kFusedWarps);
  for (int j = 0; j < g.n_can; ++j) {
    int e0 = g.seg_start[j], e1 = g.seg_start[j + 1];
    while (e0 < e1 && (g.src[e0] >> 1) < lo) ++e0;
    int e2 = e0;
    while (e2 < e1 && (g.src[e2] >> 1) < hi) ++e2;
    const int n = e2 - e0;
    if (n == 0) continue;
    const int n_pieces = (n + kFusedLcap - 1) / kFusedLcap;
    int first = e0;
    for (int q = 0; q < n_pieces; ++q) {
      const int len = n / n_pieces + (q < n % n_pieces ? 1 : 0);
      pieces[owner[j]].push_back({len, slot[j], first});
      first += len;
    }
  }
  std::vector<unsigned char> &o = out.bytes;
  o.assign(128, 0);
  static const int perms[24][4] = {{0,1,2,3},{0,1,3,2},{0,2,1,3},{0,2,3,1},{0,3,1,2},{0,3,2,1},{1,0,2,3},{1,0,3,2},
                                   {1,2,0,3},{1,2,3,0},{1,3,0,2},{1,3,2,0},{2,0,1,3},{2,0,3,1},{2,1,0,3},{2,1,3,0},
                                   {2,3,0,1},{2,3,1,0},{3,0,1,2},{3,0,2,1},{3,1,0,2},{3,1,2,0},{3,2,0,1},{3,2,1,0}};
  for (int w = 0; w < kFusedWarps; ++w) {
    auto &pw = pieces[w];
    std::stable_sort(pw.begin(), pw.end(), [](const FusedPiece &a, const FusedPiece &b) { return a.len > b.len; });
    std::vector<PackGroup> groups;
    constexpr int thresh = 99;               // a spare group is never opened for a colliding piece (measured: no gain)
    const int max_groups = ((int)pw.size() + 31) / 32;
    for (const FusedPiece &pc : pw) {
      int bank[kFusedLcap];
      for (int k = 0; k < pc.len; ++k) bank[k] = ((g.src[pc.first + k] >> 1) - lo) & 15;   // buffers are 128-byte aligned
      int best_cost = 1 << 30, best_g = -1, best_h = 0, best_perm = 0;
      for (int gi = 0; gi < (int)groups.size() && best_cost > 0; ++gi) {
        PackGroup &G = groups[gi];
        if (std::find(G.cells.begin(), G.cells.end(), pc.slot) != G.cells.end()) continue;
        for (int h = 0; h < 2 && best_cost > 0; ++h) {
          if (G.n[h] >= 16) continue;
          const int sc = 2 * G.scount[h][pc.slot & 15];
          for (int pi = 0; pi < 24; ++pi) {
            // the piece's k-th visibility goes to row perms[pi][k]; rows must be < L and distinct
            bool valid = true;
            int cost = sc;
            for (int k = 0; k < pc.len; ++k) {
              const int r = perms[pi][k];
              if (r >= G.L) { valid = false; break; }
              cost += G.bcount[h][r][bank[k]];
            }
            if (valid && cost < best_cost) { best_cost = cost; best_g = gi; best_h = h; best_perm = pi; }
            if (best_cost == 0) break;
          }
        }
      }
      // no free lane anywhere, or only badly colliding ones while a spare group is allowed: a new
      // group, as long as this piece
      if (best_g < 0 || (best_cost >= thresh && (int)groups.size() < max_groups)) {
        PackGroup G;
        G.L = pc.len;
        std::fill(&G.lane_slot[0], &G.lane_slot[32], -1);
        for (auto &le : G.lane_entry) std::fill(&le[0], &le[kFusedLcap], -1);
        groups.push_back(G);
        best_g = (int)groups.size() - 1; best_h = 0; best_perm = 0;
      }
      PackGroup &G = groups[best_g];
      const int lane = best_h * 16 + G.n[best_h]++;
      G.cells.push_back(pc.slot);
      G.lane_slot[lane] = pc.slot;
      G.scount[best_h][pc.slot & 15]++;
      G.sbank[best_h] |= 1u << (pc.slot & 15);
      for (int k = 0; k < pc.len; ++k) {
        const int r = perms[best_perm][k];
        G.lane_entry[lane][r] = pc.first + k;
        G.bcount[best_h][r][bank[k]]++;
      }
    }
    std::stable_sort(groups.begin(), groups.end(), [](const PackGroup &a, const PackGroup &b) { return a.L > b.L; });
    if ((int)groups.size() > kFusedMaxGroups) { ok = false; return; }
    uint32_t lseq = 0;                     // groups per length class, L = 4 in the low byte (they are sorted by L)
    for (size_t gi = 0; gi < groups.size(); ++gi) lseq += 1u << (8 * (kFusedLcap - groups[gi].L));
    const uint32_t off = (uint32_t)o.size() | ((uint32_t)groups.size() << 24);
    std::memcpy(o.data() + 8 * w, &off, 4);
    std::memcpy(o.data() + 8 * w + 4, &lseq, 4);
    for (const PackGroup &G : groups) {
      const size_t base = o.size();
      o.resize(base + (size_t)(G.L + 1) * 64, 0);
      uint16_t *rows = reinterpret_cast<uint16_t *>(o.data() + base);
      out.groups++;
      out.rows += G.L;
      out.warp_cost[w] += kGroupCost + kRowCost * G.L;
      for (int h = 0; h < 2; ++h) {
        int mx = 1;
        for (int bk = 0; bk < 16; ++bk) mx = std::max(mx, G.scount[h][bk]);
        out.rmw_wavefronts += mx;
        for (int r = 0; r < G.L; ++r) {
          int m = 1;
          for (int bk = 0; bk < 16; ++bk) m = std::max(m, G.bcount[h][r][bk]);
          out.halfrow_wavefronts += m;
        }
        // empty lanes fold zero into the zero slot of a bank the half does not use
        int fb = 0;
        for (int l = h * 16; l < h * 16 + 16; ++l) {
          if (G.lane_slot[l] >= 0) { rows[l] = (uint16_t)G.lane_slot[l]; continue; }
          while (fb < 15 && (G.sbank[h] >> fb & 1u)) ++fb;
          rows[l] = (uint16_t)(sink0 + fb);
          if (fb < 15) ++fb;
        }
      }
      for (int l = 0; l < 32; ++l)
        for (int r = 0; r < G.L; ++r) {
          uint16_t e = 0x7FFFu;
          if (G.lane_entry[l][r] >= 0) {
            const int code = g.src[G.lane_entry[l][r]];
            e = (uint16_t)(((code >> 1) - lo) | ((code & 1) << 15));
          }
          rows[(size_t)(r + 1) * 32 + l] = e;
        }
    }
  }
  o.resize((o.size() + 15) / 16 * 16, 0);
}

// cell -> warp: longest first to the least loaded warp; the cells of a warp get consecutive slots
// of S in that order, so their banks cycle
static void assign_cells(const HostGather &g, std::vector<int> &owner, std::vector<int> &slot) {
  std::vector<int> order(g.n_can);
  for (int j = 0; j < g.n_can; ++j) order[j] = j;
  auto len = [&](int j) { return g.seg_start[j + 1] - g.seg_start[j]; };
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return len(a) > len(b); });
  std::vector<long> load(kFusedWarps, 0);
  constexpr int w0bias = 4;                  // percent of a warp's share
  load[0] = (long)g.n_kept * w0bias / (100 * kFusedWarps);     // warp 0 also runs the chunk ring (thread 0)
  owner.assign(g.n_can, 0);
  for (int j : order) {
    const int w = (int)(std::min_element(load.begin(), load.end()) - load.begin());
    owner[j] = w;
    load[w] += len(j) + 2;            // + the cost of folding the group sum into S[j]
  }
  slot.assign(g.n_can, 0);
  int next = 0;
  for (int w = 0; w < kFusedWarps; ++w)
    for (int j : order)
      if (owner[j] == w) slot[j] = next++;
}

// relative entries -> shared-memory slots of the buffer the chunk will land in (base_slot, in
// 8-byte units); a padded entry reads the zero slot of a bank that the real entries of its
// half-row leave free
// (zslot0: first of 16 consecutive always-zero slots a padded visibility entry may point at -- the sinks in
// S, or, when correction factors ride along, 16 slots whose partners f_off behind them are finite too)
static void finalize_chunk_table(std::vector<unsigned char> &b, uint32_t base_slot, uint32_t zslot0) {
  for (int w = 0; w < kFusedWarps; ++w) {
    uint32_t off, lseq;
    std::memcpy(&off, b.data() + 8 * w, 4);
    std::memcpy(&lseq, b.data() + 8 * w + 4, 4);
    size_t blk = off & 0xFFFFFFu;
    for (int gi = 0; gi < (int)(off >> 24); ++gi) {
      const int L = group_len(lseq, gi);
      uint16_t *rows = reinterpret_cast<uint16_t *>(b.data() + blk);
      for (int r = 1; r <= L; ++r)
        for (int half = 0; half < 2; ++half) {
          uint16_t *e = rows + (size_t)r * 32 + half * 16;
          uint32_t used = 0;
          for (int l = 0; l < 16; ++l)
            if ((e[l] & 0x7FFFu) != 0x7FFFu) {
              const uint32_t sl = base_slot + (e[l] & 0x7FFFu);
              e[l] = (uint16_t)(sl | (e[l] & 0x8000u));
              used |= 1u << (sl & 15);
            } else {
              e[l] = 0xFFFFu;                                             // marks padding until the bank is chosen
            }
          int free_bank = 0;
          while (free_bank < 15 && (used >> free_bank & 1u)) ++free_bank;
          for (int l = 0; l < 16; ++l)
            if (e[l] == 0xFFFFu) e[l] = (uint16_t)(zslot0 + ((free_bank - (int)zslot0) & 15));
        }
      blk += (size_t)(L + 1) * 64;
    }
  }
}


}  // namespace blink
