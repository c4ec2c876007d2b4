// Kernel argument block of the dense (tensor-pipe) sa_run kernel (sa_dense_kernel.cu).
// Included by the host code AND prepended to the kernel source that NVRTC compiles, so it uses
// only built-in types.  Plain data, device pointers.
#ifndef TSA_DENSE_PARAMS_H
#define TSA_DENSE_PARAMS_H

namespace tsa_dense {

typedef unsigned int u32;
typedef unsigned short u16;
typedef unsigned long long u64;
typedef long long i64;
typedef signed char i8;

// wloc word of edge e: bits 0-7 A-fragment register, 8-9 byte in it, 10-14 lane, 16-31 slot (byte
// offset of the weight in the chain's canonical weight row).
// thloc word of node i: bits 0-2 thread group g (lane / 4), 3-4 threshold word w, 5-6 byte j,
// 16-31 entry (byte offset of the pair index in the chain's canonical threshold row).
struct Params {
  // problem tables (one per problem, shared by all chains)
  const u16* frag_slot;   // [MT*KS*4][32][4] canonical weight-row offset feeding each A-fragment byte, 0xFFFF = structural zero
  const u32* meta;        // [tiles][32] sparse layout: selector word of each A tile, per lane
  const u16* th_entry;    // [8][NW][4]        canonical threshold-row offset of the node in (group g, word w, byte j), 0xFFFF = padding row
  const u32* init_frag;   // [32][2*KS]        B fragments of the t = 0 states, per lane
  const u32* obs_word;    // [NOBS][32][NW][2] observed values in the layout of a lane's result words (3 = not scored)
  const u32* fix;         // [NFIX_ROUNDS][32] clamp fix-ups: bits 0-15 byte offset in the state buffer, 16-17 value, bit 31 valid
  const u32* wloc;        // [E]
  const u32* thloc;       // [N]
  // structural constraints (kernels built with TSD_CONSTRAINED=1): CSR over the nodes' in- / out-edges holding each
  // edge's offset in the canonical weight row, and the end points of every caller edge (src | dst << 16)
  const int* con_in_ptr;  // [N+1]
  const int* con_in_slot; // [E]
  const int* con_out_ptr; // [N+1]
  const int* con_out_slot;// [E]
  const u32* edge_nodes;  // [E]
  i8 tha[16];             // -t_lo     per threshold pair
  i8 thb[16];             // -t_hi - 1 per threshold pair
  int fit_const;          // mismatches of clamped observed entries minus the always-counted unscored entries
  // chain store (HBM, SoA; same canonical rows as the other kernel families)
  int R;
  i8* cur_w;              // [R][EPADA]
  i8* cur_th;             // [R][NPADA]
  i8* best_w;
  i8* best_th;
  u32* fit_cur;           // [R]
  u32* fit_best;
  // annealing schedule
  u32 key0, key1, chain_id_base;
  int n_levels, dmax;
  i64 steps_per_level;
  const u32* accept;      // [L][D]
  // trace (row == nullptr: off)
  const int* trace_row;   // [R]
  u64* trace_rec;         // [n][trace_max]
  i64 trace_max;
  u64 trace_g0;
  // acceptance statistics per temperature level (nullptr: off): [L][4] = steps, accepted, accepted worse, new best
  u64* level_stats;
  // this launch
  u64 g0;
  i64 steps;
  // balanced slots (0 = one chain per slot): every slot advances slot_steps chain-steps of the line
  // of R*steps; flags[chain] != 0 once the head piece of a straddling chain is back in HBM
  i64 slot_steps;
  u32* flags;             // [R], zeroed by the host before the launch
  u32* err;               // [1] set to 1 if a hand-over wait gave up (the launch's results are then invalid)
};

}  // namespace tsa_dense
#endif
