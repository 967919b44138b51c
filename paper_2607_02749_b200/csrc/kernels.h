// kernels.h -- host-callable launchers of the sm_100a kernels (kernels.cu).  All pointers are DEVICE pointers into
// the caller's workspace unless stated otherwise; every launcher enqueues on `stream` and returns the CUDA error
// of the launch (0 = success).  `launches` is incremented by the number of kernels enqueued.
#pragma once
#include <stddef.h>
#include <stdint.h>

#include "devprog.h"

namespace gv {

struct TileDesc { uint8_t k, n_runs, pad[2]; Run runs[MAX_RUNS]; };

struct GateLaunch {
    const DBlock *blocks; const DStage *stages; const DOp *ops; const DSeg *segs; const DTrz *trzs;
    const uint64_t *tczs; const int32_t *csidx; const int16_t *ryl; const DCx *cxs; const uint32_t *slut;
};

constexpr uint32_t EXPECT_TAB_CAP = 2048;   // complex entries of the shared-memory W-table area
constexpr int EXPECT_UMAX = 8;              // largest single table: 2^8 entries
constexpr uint32_t READOUT_BLOCKS = 148 * 8;   // grid of the read-out sweep: 8 blocks of 256 threads per SM
constexpr int SAMPLE_CHUNK_LOG2 = 12;            // shot sampling: probability mass is tabulated per 4096 amplitudes
constexpr uint32_t SAMPLE_MAX_SHOTS = 1u << 16; // shots per gvqe_sample call (uniforms and results staged in the workspace)
constexpr uint32_t SWEEP_MAX_ROWS = 1u << 14;   // rows of one parameter-shift sweep staged in the workspace (codes in, energies out)
constexpr uint32_t HDR_BYTES = 384;         // shared-memory header of the gate kernel
constexpr uint32_t EXPECT_HDR_BYTES = 1024; // shared-memory header of the expectation kernel: holds the DPass copy

struct PrefixDev {   // device view of schedule.h Prefix
    const int32_t *rot_begin; const uint8_t *rot_kind; const int32_t *rot_param;
    const uint8_t *cx_t, *cx_c;
    int n_cx, n_cz, n, kk;   // kk: log2 of the amplitudes one thread block writes (contiguous)
    int cz_d[4];
    uint64_t cz_m[4];
    // x = A^-1 y inside one thread block of 2^kk amplitudes: vary = the x bits that differ among them (n_vary <= 40 of them,
    // numbered in ascending order: vq[j] = the j-th), cimg[b] = image of offset bit b < kk as a compact index over those bits
    uint64_t vary;
    int n_vary;
    uint8_t vq[40];
    uint64_t cimg[16];
};

// prec: 0 = complex64 (float), 1 = complex128 (double)
// ry: optional second table for the specialised gate kernels ({tan, scale, form, 0} per parameter, jit.cpp), or NULL
int launch_expand_params(int prec, const double *params, void *cs, void *ry, uint64_t count, void *stream, uint64_t *launches);
// rows[r][:] = theta[:] with (code[r] & 1 ? -pi/2 : +pi/2) added to parameter code[r] >> 1 (all DEVICE pointers)
int launch_shift_rows(const double *theta, const int32_t *code, double *rows, int P, int n_rows, void *stream, uint64_t *launches);
int launch_init_product(int prec, const PrefixDev &pd, void *states, uint64_t stride_amps, const void *cs, int P, int batch,
                        void *stream, uint64_t *launches);
int launch_gate_block(int prec, int R, const GateLaunch &g, const DBlock &block, int k, uint32_t smem_prog_bytes, int n,
                      void *states, uint64_t stride_amps, const void *cs, int P, int batch, void *stream,
                      uint64_t *launches);
int launch_expect_pass(int prec, const DPass *passes, int pass_index, int k, int n, const DGroup *groups,
                       const DTerm *terms, const void *wstat, const uint32_t *gtabs, const DRs *rss, const void *states, uint64_t stride_amps, const void *table, double *partial,
                       uint32_t slots_per_b, uint32_t slot_off, int batch, void *stream, uint64_t *launches);
int launch_reduce(double *partial, uint32_t slots_per_b, double *E, int batch, void *stream, uint64_t *launches);
int launch_table_scatter(int prec, void *table, const uint64_t *z, const double *c, uint32_t count, void *stream,
                         uint64_t *launches);
int launch_fwht_pass(int prec, void *table, const TileDesc &td, uint32_t bitmask, int n, void *stream, uint64_t *launches);
// Most probable basis state of `count` amplitudes; scratch: (READOUT_BLOCKS + 1) * 16 bytes, result {double p, uint64 x} at [0].
int launch_argmax(int prec, const void *state, uint64_t count, void *scratch, void *stream, uint64_t *launches);
// The same sweep with its per-block entries in a file-scope device array (kernels.cu): no allocation, no context.
// result (DEVICE): {double p, uint64 x}.  Returns a cudaError_t value (0 = launched).
constexpr size_t NOALLOC_SCRATCH_BYTES = 32 * 1024;       // >= READOUT_BLOCKS entries of 16 bytes
constexpr uint64_t NOALLOC_MAX_AMPLITUDES = 1ull << 34;   // largest statevector the entry point takes
int launch_argmax_noalloc(int prec, const void *state, uint64_t count, void *result, void *stream);
// Inverse-CDF sampling: mass = ceil(count / 2^SAMPLE_CHUNK_LOG2) doubles (becomes the exclusive prefix), total = 1 double,
// u_dev = n_shots uniforms in [0,1), x_dev = n_shots results.
int launch_sample(int prec, const void *state, uint64_t count, double *mass, double *total, const double *u_dev,
                  uint64_t *x_dev, uint32_t n_shots, void *stream, uint64_t *launches);
// dst = (H or H S^dagger on qubit q) src over 2^n amplitudes (measurement basis of an X / Y letter); src may equal dst
int launch_basis_rotate(int prec, const void *src, void *dst, int n, int q, int is_y, void *stream, uint64_t *launches);
int kernels_init(void);   // opt-in shared memory sizes; returns the CUDA error

}  // namespace gv
