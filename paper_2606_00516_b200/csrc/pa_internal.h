// Internal structures shared by the host planner and the device kernels of libpa_b200.so.
// (Product code: nothing here is shared with oracle/.)
#pragma once
#include <cstdint>

namespace pa {

constexpr int kBlock = 16;          // KV block size b (tokens)
constexpr int kDecodeWarps = 8;     // persistent decode workers (warps) per CTA
constexpr int kMaxGroup = 8;        // max q heads per KV head (N of the decode MMA)
constexpr int kQTile = 128;         // prefill query-tile rows
constexpr int kKvTile = 128;        // prefill KV-tile keys

// One decode work item: a run of whole KV blocks of one (decode sequence, KV head).
// "(seq, kv head, kv chunk)".
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
    int32_t* queue;            // [0] next decode bundle, [1] exited CTAs, [2] next prefill unit (all self-resetting)
    int32_t* group_counters;   // [num_decode_seqs * Hkv] arrivals of split groups (self-resetting)
    const DecItem* items;      // decode items in bundle order
    const int32_t* bundle_start; // [n_bundles + 1] item index ranges
    const PreTile* tiles;      // prefill tiles
    float2* part_ml;           // [slots][kMaxGroup] (m in log2 domain, l)
    float* part_o;             // [slots][G][D] unnormalised partial outputs
    int32_t n_items, n_bundles, n_tiles, n_split;
    int32_t n_units;           // prefill work units = n_tiles * Hkv * head_groups (tcgen05 path; 0 = none)
    int32_t head_groups;       // ceil(G / q-tiles per CTA): units per (tile, KV head)
};

}  // namespace pa
