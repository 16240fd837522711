// tile_tables.hpp -- host-side construction of the site tiles of the thread-block-cooperative fp16 hop kernel
// (hop_tile.cuh).  No CUDA.
//
// Why tiles: an 8-neighbour stencil without on-chip reuse pulls every input column through L2 -> SM eight times; at
// Ls = 16 that is 8 x 768 B per output column and the kernel sits on the L2 slice throughput, not on HBM (DESIGN.md
// section 4).  A tile is a set of at most TS output sites of one stage list chosen compact in 4D (a 4x4x2x2 cell of one
// parity holds 32 sites whose 256 neighbour references hit only 128 distinct input columns), so each distinct input
// column is staged once per tile in shared memory and read from there by all output sites that need it.
//
// The tables are geometry only (shared by all Dirichlet blocks, independent of Ls and of the gauge field):
//   out_site[j]   list index of the j-th output site of the tile
//   slot[j][d]    shared-memory slot (index into in_col) of the neighbour in direction d (NIN, a column of zeros, where absent)
//   have[j]       bit d set <=> neighbour d exists (inside the Dirichlet pad box and below the input limit of the stage)
//   in_col[i]     list index (in the stage's input list) of the i-th staged input column (ascending; in_run marks the runs
//                 of consecutive columns, each fetched by one bulk copy; out_run the runs of consecutive output sites)
#pragma once
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <unordered_map>
#include <vector>

namespace mspcg {

constexpr int TILE_TS = 32;     // output sites per tile
constexpr int TILE_NIN = 128;   // staged input columns per tile

struct TileRec {                // 1104 bytes, 16-byte aligned; the first TILE_HDR bytes are staged for the consumer warps
  int n_out, n_in, pad0, pad1;  // pad0: 1 if every site of the tile has all eight neighbours
  int out_site[TILE_TS];        // ascending
  uint8_t slot[TILE_TS][8];
  uint8_t have[TILE_TS];
  int in_col[TILE_NIN];         // ascending: slot i holds input column in_col[i]
  uint8_t in_run[TILE_NIN];     // in_run[i] = n > 0: in_col[i .. i+n) are consecutive columns, fetched by ONE copy into slots i .. i+n
  uint8_t out_run[TILE_TS];     // the same for the output sites (their link records are consecutive in memory)
};
constexpr int TILE_HDR = 16 + TILE_TS * 4 + TILE_TS * 8 + TILE_TS;   // 432
static_assert(sizeof(TileRec) == TILE_HDR + TILE_NIN * 5 + TILE_TS, "TileRec layout");
static_assert(sizeof(TileRec) % 16 == 0 && TILE_HDR % 16 == 0, "TileRec alignment");

// Tiles over the output sites [lo, hi) of a stage list with coordinates coords[n][4] and neighbour table nbr[n][8]
// (indices into the input list, -1 = absent); neighbours >= in_limit are dropped (kernel 2 of a Dirichlet block reads
// only the block-interior sites of its input).  Sites are taken cell by cell (the 4x4x2x2 cells of geometry.hpp, so in list
// order inside each of the two parts of a list) and packed greedily: a tile is closed when it has TS sites or would need
// more than NIN input columns.
inline std::vector<TileRec> build_tiles(const std::vector<short>& coords, const std::vector<int>& nbr, int lo, int hi, int in_limit) {
  std::vector<TileRec> tiles;
  if (hi <= lo) return tiles;
  const int cell[4] = {4, 4, 2, 2};
  std::vector<std::pair<uint64_t, int>> order;
  order.reserve(hi - lo);
  for (int i = lo; i < hi; i++) {
    uint64_t key = 0;
    for (int d = 3; d >= 0; d--) key = (key << 12) | (uint64_t)(((int)coords[4 * (size_t)i + d] + 4) / cell[d]);
    order.emplace_back(key, i);
  }
  std::sort(order.begin(), order.end());
  std::vector<int> members;
  std::unordered_map<int, int> slot_of;
  auto close = [&]() {
    if (members.empty()) return;
    TileRec cur; memset(&cur, 0, sizeof(cur));
    std::sort(members.begin(), members.end());
    std::vector<int> cols; cols.reserve(slot_of.size());
    for (const auto& kv : slot_of) cols.push_back(kv.first);
    std::sort(cols.begin(), cols.end());
    cur.n_in = (int)cols.size();
    for (int i = 0; i < cur.n_in; i++) { cur.in_col[i] = cols[i]; slot_of[cols[i]] = i; }
    for (int i = 0; i < cur.n_in;) { int n = 1; while (i + n < cur.n_in && cols[i + n] == cols[i] + n) n++; cur.in_run[i] = (uint8_t)n; i += n; }
    cur.n_out = (int)members.size();
    memset(cur.slot, TILE_NIN, sizeof(cur.slot));   // absent neighbours read the zero column
    for (int j = 0; j < cur.n_out; j++) {
      const int i = members[j];
      cur.out_site[j] = i;
      for (int d = 0; d < 8; d++) {
        const int nb = nbr[(size_t)i * 8 + d];
        if (nb < 0 || nb >= in_limit) continue;
        cur.slot[j][d] = (uint8_t)slot_of[nb];
        cur.have[j] |= (uint8_t)(1u << d);
      }
    }
    for (int j = 0; j < cur.n_out;) { int n = 1; while (j + n < cur.n_out && members[j + n] == members[j] + n) n++; cur.out_run[j] = (uint8_t)n; j += n; }
    cur.pad0 = 1;   // flag: every site of the tile has all eight neighbours
    for (int j = 0; j < cur.n_out; j++) if (cur.have[j] != 0xff) cur.pad0 = 0;
    tiles.push_back(cur);
    members.clear(); slot_of.clear();
  };
  for (const auto& kv : order) {
    const int i = kv.second;
    int fresh = 0;
    int seen[8]; int nseen = 0;
    for (int d = 0; d < 8; d++) {
      const int nb = nbr[(size_t)i * 8 + d];
      if (nb < 0 || nb >= in_limit || slot_of.count(nb)) continue;
      bool dup = false;
      for (int q = 0; q < nseen; q++) dup = dup || seen[q] == nb;
      if (!dup) { seen[nseen++] = nb; fresh++; }
    }
    if ((int)members.size() == TILE_TS || (int)slot_of.size() + fresh > TILE_NIN) close();
    members.push_back(i);
    for (int d = 0; d < 8; d++) {
      const int nb = nbr[(size_t)i * 8 + d];
      if (nb >= 0 && nb < in_limit) slot_of.emplace(nb, 0);
    }
  }
  close();
  return tiles;
}

// Host-side check of a tiling against the neighbour table it was built from: every output site of [lo, hi) in exactly one tile, every
// present neighbour's slot holding exactly that neighbour's column, absent ones pointing at the zero column with their presence bit clear,
// input columns ascending and distinct, copy runs covering every slot exactly once with consecutive columns.  Returns 0 or a failure code.
inline int check_tiles(const std::vector<TileRec>& tiles, const std::vector<int>& nbr, int lo, int hi, int in_limit) {
  std::vector<char> seen(hi > lo ? hi - lo : 0, 0);
  for (const TileRec& t : tiles) {
    if (t.n_out < 1 || t.n_out > TILE_TS || t.n_in < 0 || t.n_in > TILE_NIN) return 1;
    for (int i = 1; i < t.n_in; i++) if (t.in_col[i] <= t.in_col[i - 1]) return 2;
    int covered = 0;
    for (int i = 0; i < t.n_in;) {
      const int n = t.in_run[i];
      if (n < 1 || i + n > t.n_in) return 3;
      for (int q = 1; q < n; q++) if (t.in_run[i + q] != 0 || t.in_col[i + q] != t.in_col[i] + q) return 4;
      covered += n; i += n;
    }
    if (covered != t.n_in) return 5;
    for (int j = 0; j < t.n_out;) {
      const int n = t.out_run[j];
      if (n < 1 || j + n > t.n_out) return 6;
      for (int q = 1; q < n; q++) if (t.out_run[j + q] != 0 || t.out_site[j + q] != t.out_site[j] + q) return 7;
      j += n;
    }
    bool full = true;
    for (int j = 0; j < t.n_out; j++) {
      const int site = t.out_site[j];
      if (site < lo || site >= hi || seen[site - lo]) return 8;
      seen[site - lo] = 1;
      for (int d = 0; d < 8; d++) {
        const int nb = nbr[(size_t)site * 8 + d];
        const bool present = nb >= 0 && nb < in_limit;
        if (present != (((t.have[j] >> d) & 1) != 0)) return 9;
        if (present) { if (t.slot[j][d] >= t.n_in || t.in_col[t.slot[j][d]] != nb) return 10; }
        else { if (t.slot[j][d] != TILE_NIN) return 11; full = false; }
      }
    }
    if ((t.pad0 != 0) != full) return 12;
  }
  for (char c : seen) if (!c) return 13;
  return 0;
}

// staged input columns per output site (8 without reuse): the figure of merit of a tiling
inline double tiles_inputs_per_output(const std::vector<TileRec>& t) {
  long in = 0, out = 0;
  for (const TileRec& r : t) { in += r.n_in; out += r.n_out; }
  return out ? (double)in / (double)out : 0.0;
}

}  // namespace mspcg
