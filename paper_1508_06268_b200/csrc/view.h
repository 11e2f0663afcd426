// view.h -- the device-side view of one handle's state, passed by value to every kernel.
//
// HBM layout.  int8 mode: one byte per spin holding 0 (down) or 1 (up),
// colour-separated: for realisation d and slot r the two checkerboard colours are stored as
//   spins[((d*R + r)*2 + c)*Nh + j],   j = xh + Lh*(y + L*z),  x = 2*xh + ((y+z+c)&1),  Lh = L/2,
// so j is exactly the same-colour site index that keys the Philox counter, four consecutive j
// (one 32-bit word) share one Philox call, and all six neighbours of a colour-c site live in the
// other colour's array at the same (y,z,xh), at xh-1+2*parity, and at y+-1 / z+-1 with the same xh.
#pragma once
#include <cstdint>

namespace rfim {

struct GaussEntry { float x, y; };   // arg = fma((float)g_i, y, x): log2 of the acceptance probability, + 32

struct View {
    int L, Lh, R, n, D, kind;
    int W;                         // 32-bit words per row per colour (L/8), 0 if L % 8 != 0
    long long N, Nh;
    uint8_t* spins;                // [D][R][2][Nh]
    const uint8_t* fieldb;         // bimodal: [D][2][Nh], 0x10 where h_i = +1, 0 where h_i = -1
    const float* fielda;           // Gaussian: [D][2][Nh], (float)g_i (exact: |g_i| <= 2^23)
    const int32_t* fieldg;         // Gaussian: [D][2][Nh], g_i
    const uint32_t* etab;          // bimodal: [D][R(rank)][32], thr - 1 (accept iff u <= e), idx = n1 | s<<3 | hb<<4
    const uint32_t* never;         // bimodal: [D][R(rank)], bit idx set where thr = 0
    const GaussEntry* gtab;        // Gaussian: [D][R(rank)][16], idx = n1 | s<<3
    const float* band;             // Gaussian: [D][R(rank)], half-width of the float-path guard band
    const double* beta;            // [D][R(rank)]
    int32_t* t2r;                  // [D][R]
    int32_t* r2t;                  // [D][R]
    const uint32_t* keys;          // [D][2]
    long long* acc;                // [D][R(slot)][3]: Eb, Ef, Msum accumulators of the reduction
    long long* last;               // [D][R(slot)][3]: the terms the last exchange step consumed (acc is zeroed by it)
    double* ework;                 // [D][R(rank)] energies of the current exchange step
    unsigned long long* att;       // [D][R]
    unsigned long long* accn;      // [D][R]
    long long* series;             // [capacity][D][R(rank)][3]
    unsigned long long* diag;      // [4], see rfim_pt_get_diagnostics
    double J, hs;                  // hs = h (bimodal) or h * 2^-20 (Gaussian)
    int packed;                    // != 0: `spins` holds one BIT per spin (bit j & 7 of byte j >> 3, same index j as the byte layout)
    // Replica sharding: this handle STORES Rs slots of every member, slot0 + j * sstride for
    // j = 0 .. Rs-1 (all R of them when shard == 0: slot0 = 0, sstride = 1; a contiguous window: sstride = 1; a round-robin
    // deal over G ranks: slot0 = rank, sstride = G), and a sweep visits n_it replicas: every rank t < n
    // (shard == 0) or the first n_it stored slots, the active ones (shard != 0).  t2r, r2t, tables, acc, series stay global
    // (indexed by rank / slot < R).
    int shard, slot0, Rs, n_it, sstride;
    __host__ __device__ int stored_slot(int j) const { return slot0 + j * sstride; }                     // j-th stored slot
    __host__ __device__ bool stores(int slot) const { return slot >= slot0 && (slot - slot0) % sstride == 0 && (slot - slot0) / sstride < Rs; }
    __host__ __device__ int stored_index(int slot) const { return (slot - slot0) / sstride; }
};

}  // namespace rfim
