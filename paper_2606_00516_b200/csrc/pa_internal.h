// Internal structures shared by the host planner and the device kernels of libpa_b200.so.
// (Product code: nothing here is shared with oracle/.)
#pragma once
#include <cstdint>

namespace pa {

constexpr int kBlock = 16;          // KV block size b (tokens)
constexpr int kDecodeWarps = 8;     // persistent decode workers (warps) per CTA
constexpr int kMaxGroup = 8;        // max q heads per KV head (N of the decode MMA)
constexpr int kQTile = 128;         // prefill query-tile rows

// One decode work item: a run of whole KV blocks of one (decode sequence, KV head).
// "(seq, kv head, kv chunk)".  Items are not stored in HBM: the producer lane of a stream derives
// them from its bundle descriptor (below) and context_lens, and hands them to the consumer warp through shared memory.
struct DecItem {
    int32_t seq;        // sequence index in the batch
    int32_t kv_head;    // KV head g
    int32_t blk_begin;  // first logical block of the run
    int32_t blk_end;    // one past the last logical block
    int32_t kv_len;     // ctx + 1: keys [0, kv_len) are visible; the run covers keys [16*blk_begin, min(16*blk_end, kv_len))
    int32_t part_base;  // first partial slot of this (seq, kv head) group, -1 if the group is not split
    int32_t part_idx;   // this item's index among the group's parts
    int32_t n_parts;    // parts of the group (1 = write the output row directly)
};
static_assert(sizeof(DecItem) == 32, "DecItem layout");

// One decode bundle: a contiguous run of the block stream formed by all (decode sequence, KV head) groups in
// group order (group id = seq * Hkv + kv head).  It starts at block `blk_begin` of group `grp_begin` and ends with
// block `blk_end - 1` of group `grp_end` (blk_end < 0: the group's last block); every group strictly between the two
// is covered whole.  A group that a bundle boundary cuts is a split group: its parts write partials into slots
// part_base + part_idx and the last-arriving part merges them.  Only the first and the last group of a bundle can be
// split (part_base < 0: not split).  The planner writes O(bundles) of these instead of O(groups) items.
struct DecBundle {
    int32_t grp_begin, blk_begin, grp_end, blk_end;
    int32_t first_part_base, first_part;   // first group: slot base, (part_idx << 16) | n_parts
    int32_t last_part_base, last_part;     // last group (when grp_end > grp_begin): the same
};
static_assert(sizeof(DecBundle) == 32, "DecBundle layout");

// One prefill tile: up to kQTile consecutive query rows of one prefill chunk (all heads handled by the kernel grid).
struct PreTile {
    int32_t seq;       // sequence index
    int32_t q_begin;   // first query (within the chunk) of the tile
    int32_t q_rows;    // rows in the tile (<= kQTile)
    int32_t ctx;       // cached tokens before the chunk: query j sees keys 0 .. ctx + j
    int32_t kv_len;    // ctx + q_len of the whole chunk (slots at positions >= kv_len hold nothing)
    int32_t row0;      // cu_seqlens_q[seq]: first packed token row of the chunk
    int32_t pad[2];
};
static_assert(sizeof(PreTile) == 32, "PreTile layout");

// Device-side view of the planned workspace (all pointers into the caller's workspace buffer).
struct PlanView {
    int32_t* queue;            // [0] next decode bundle, [1] exited CTAs, [2] next prefill unit, [3] rows to redo (all self-resetting), [4] rows redone since pa_plan
    int32_t* group_counters;   // [num_decode_seqs * Hkv] arrivals of split groups (self-resetting)
    const DecBundle* bundles;  // [n_bundles] decode bundles
    int2* redo;                // prefill rows whose one-pass softmax overflowed: {tile index, (row in tile << 8) | q head}
    const PreTile* tiles;      // prefill tiles
    float2* part_ml;           // [slots][kMaxGroup] (m in log2 domain, l)
    float* part_o;             // [slots][G][D] unnormalised partial outputs
    int32_t n_items, n_bundles, n_tiles, n_split;
    int32_t n_units;           // prefill work units = n_tiles * Hkv * head_groups (tcgen05 path; 0 = none)
    int32_t head_groups;       // ceil(G / q-tiles per CTA): units per (tile, KV head)
    // Guided hand-out of decode bundles: a bundle of n groups is taken in n_levels pieces, piece l = the groups
    // [n * cum[l] / 256, n * cum[l + 1] / 256) of the bundle (cum[0] = 0, cum[n_levels] = 256; cum[1..8] packed one byte
    // each into level_cum).  The queue hands out tickets = level * n_bundles + bundle, level-major, so every stream
    // starts with the large first piece of its own bundle and the small late pieces even out unequal stream rates at
    // no cost to the planner and without cutting any more groups.  n_levels = 1: a ticket is a whole bundle.
    int32_t n_levels;
    uint64_t level_cum;
};

}  // namespace pa
