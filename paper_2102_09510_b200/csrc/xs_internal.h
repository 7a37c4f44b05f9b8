// xs_internal.h -- declarations shared by the translation units of libxs_b200.so.
// Product code: shares nothing with oracle/ (own Philox, own generator).
#pragma once
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/xs.h"

namespace xs {

// Domain tags in Philox counter word 3.
enum : uint32_t { TAG_GRAPH = 1, TAG_GAUGE = 2, TAG_INIT = 3, TAG_SWEEP = 4, TAG_PARTITION = 5, TAG_CLONE = 6 };

// ---- host-side instance (a-1) -------------------------------------------------------------
struct HostGraph {
    uint32_t n = 0;
    std::vector<uint32_t> tri;       // [N][3]
    std::vector<uint8_t> jbit;       // [N]
    std::vector<uint32_t> nbr;       // [N][6]  partners of spin i in its clauses (ascending clause id)
    std::vector<uint32_t> cls;       // [N][3]  clause ids of spin i
    std::vector<uint32_t> order;     // [N]
    std::vector<uint32_t> set_start; // [n_sets + 1]
    int attempt = -1;                // accepted attempt of the configuration model
};

void philox4x32_10_host(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

// Build from seeds (configuration model with rejection, gauge, adjacency, greedy or balanced sets).
// Returns false and sets err on failure.
bool build_graph_from_seed(uint32_t n, uint64_t graph_seed, bool gauge, uint32_t set_cap, bool balanced,
                           HostGraph& g, std::string& err);
// Build from explicit arrays; validates 3-regularity and that every set is an anti-clique.
bool build_graph_from_arrays(uint32_t n, const uint32_t* tri, const uint8_t* jbit,
                             const uint32_t* order, const uint32_t* set_size, uint32_t n_sets,
                             HostGraph& g, std::string& err);

// ---- device tables --------------------------------------------------------------------------
// Adjacency record of the spin at position p of the update order (32 bytes, 2 x 16 B loads).
struct alignas(16) AdjRec {
    uint32_t nbr[6];   // spin indices: (nbr[2r], nbr[2r+1]) = partners in clause r
    uint32_t self;     // spin index of this position
    uint32_t jbits;    // bit r = coupling bit of clause r (1 <=> J = -1)
};
// Clause record for the energy / ground-state kernels (16 bytes).
struct alignas(16) ClauseRec {
    uint32_t i, j, k, jbit;
};

// Task record of the clause-word kernel (xs_sweep_clause.cu): shared-memory row offsets of the
// three clause rows of the spin at entry round * n_slots + slot, and the spin index
// (0xFFFFFFFF: the slot is idle in that round and works on a scratch row) (16 bytes).
struct alignas(16) CRec {
    uint32_t off0, off1, off2, spin;
};

// Device workspace carved out of the caller's buffer.
struct DevLayout {
    size_t off_x = 0, off_first_hit = 0, off_adj = 0, off_clause = 0, off_set_start = 0,
           off_rec = 0, off_seed = 0, off_det = 0, off_nsets = 0, off_crec = 0, off_cplace = 0, off_cbar = 0, off_cthr = 0, total = 0;
};
DevLayout make_layout(const xs_params& p);
// Task-table entries per instance (CRec crec[I][entries]): 2 N, and at least 256 for batches of up
// to 1024 small instances so that the latency kernel's 16-slot passes always fit.
inline uint32_t crec_entries(const xs_params& p)
{
    const uint32_t e = 2u * p.n_spins;
    return (e < 256u && p.n_instances <= 1024u) ? 256u : e;
}

struct DevPtrs {
    uint64_t* x;           // [I][N][W]
    uint32_t* first_hit;   // [I][64W]
    AdjRec* adj;           // [I][N]   (order position)
    ClauseRec* clause;     // [I][N]
    uint32_t* set_start;   // [I][N+1]
    xs_tts_rec* rec;       // [I]
    uint64_t* run_seed;    // [I]
    uint64_t* det;         // [I][W]   scratch: OR of unsatisfied-clause words
    uint32_t* n_sets;      // [I]
    CRec* crec;            // [I][2N]  clause-word kernel: tasks, entry = round * n_slots + slot
    uint32_t* cbar;        // [I]      clause-word kernel: bit r = barrier after round r
    uint32_t* cthr;        // [2]      clause-word kernel: compare constants of the noise threshold
    uint32_t* cplace;      // [I][N]   clause-word kernel: shared-memory row offset of clause t
};

// Flip table w_0..w_3 as 32-bit thresholds: a spin with k unsatisfied
// interactions flips iff bit k of `always` is set or the word's number u < lo[k].
// general == 0: the quasi-greedy form (0, lo[1], 1, 1) -> the fast kernels apply.
struct FlipTable {
    uint32_t lo[4];
    uint32_t always;
    uint32_t general;
    // SURVEY.md 8(f) NEXT-2 (XS_FLAG_CLONE_NOISE): every clone draws its own 7-bit number U;
    // a k = 1 spin flips iff U < clone_m (w1 = clone_m / 128, 0..128)
    uint32_t per_clone;
    uint32_t clone_m;
};

struct TileGeom {
    uint32_t regime = 0;       // 0 on-chip, 1 streaming
    uint32_t T = 0;            // uint64 columns per tile
    uint32_t CW = 0;           // words per lane (1 or 2)
    uint32_t threads = 0;
    uint32_t ctas = 0;
    uint32_t smem = 0;
    uint32_t batch = 0;        // sweeps between in-kernel ground-state checks
    uint32_t rb = 0;           // sweeps of random bytes produced at a time
    uint32_t variant = 0;      // 0 generic tile kernel, 1 static-task kernel, 2 clause-word kernel
};

}  // namespace xs

struct xs_batch {
    xs_params p{};
    std::vector<xs::HostGraph> graphs;
    std::vector<uint64_t> run_seeds;
    xs::DevLayout lay;
    xs::DevPtrs d{};
    xs::TileGeom geom;
    xs::FlipTable ft{};
    uint32_t n_sets_max = 0;
    uint32_t max_set_size = 0;
    uint32_t clause_state = 0;    // clause-word kernel tables: 0 not built, 1 uploaded, 2 not eligible
    uint32_t clause_slots = 0;    // slots per CTA the uploaded tables were built for
    uint32_t clause_rounds = 0;   // rounds per sweep of those tables (4..8)
    uint64_t clause_thr = ~0ull;  // threshold the uploaded compare constants belong to
    uint32_t clause_mode = 0;
    uint32_t warp_passes = 0;     // latency kernel: passes per sweep of the uploaded tables (0 = none)     // kernel MODE the tables allow (xs_sweep_clause.cuh)
    uint64_t sweeps_issued = 0;   // upper bound on any instance's sweep counter (overflow guard)
    xs_geometry req{XS_GEOM_AUTO, 0, 0, 0, 0, 0};   // xs_set_geometry requests (0 / AUTO = rule)
    uint32_t num_sms = 148;       // cudaDevAttrMultiProcessorCount of the device the batch lives on
    int device = 0;               // CUDA device ordinal the workspace belongs to
    uint32_t flags0 = 0;          // p.flags as given by the caller (p.flags may gain XS_FLAG_STREAMING)
    void* ws = nullptr;
};

namespace xs {
// sets the thread-local message behind xs_last_error() and returns `code` (xs_api.cu)
int xs_set_error(int code, const std::string& msg);
// kernels (xs_kernels.cu); every launcher returns a cudaError_t as int.
int launch_init(const xs_batch& b, void* stream);
int launch_mark(const xs_batch& b, bool reset_first_hit, void* stream);   // ground-state marking at current t
int launch_sweeps(const xs_batch& b, uint32_t n_sweeps, void* stream);
int launch_finalize(const xs_batch& b, uint32_t n_sweeps, void* stream);
int launch_energy(const xs_batch& b, int32_t* dev_out, void* stream);
bool choose_geometry(const xs_batch& b, TileGeom& g, std::string& err);
// static-task variant (xs_sweep_static.cu)
bool static_feasible(const xs_batch& b, uint32_t T, uint32_t CW, uint32_t threads);
uint32_t static_rounds(const xs_batch& b, uint32_t T, uint32_t CW, uint32_t threads);
uint32_t static_smem_bytes(uint32_t N, uint32_t T);
int launch_sweep_static(const xs_batch& b, uint32_t n_sweeps, void* stream);
// clause-word variant (xs_sweep_clause.cu)
uint32_t clause_rounds(const HostGraph& g, uint32_t n_slots);
bool clause_placement(const HostGraph& g, uint32_t n_slots, uint32_t n_rounds, CRec* crec,
                      uint32_t* cplace, uint32_t* bar_mask, uint32_t* mode);
int clause_prepare(xs_batch& b, void* stream);
int launch_sweep_clause(const xs_batch& b, uint32_t n_sweeps, void* stream);
// latency kernel (xs_sweep_warp.cu)
int warp_prepare(xs_batch& b, void* stream);
int launch_sweep_warp(const xs_batch& b, uint32_t n_sweeps, void* stream);
}  // namespace xs
