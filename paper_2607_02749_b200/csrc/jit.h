// jit.h -- schedule-specialised gate-block kernels: CUDA C++ source generated from a compiled Program (schedule.h),
// one kernel per fused block, compiled once per context with NVRTC for sm_100a and reused by every energy call
// ("JIT-compiled once and reused across all optimization iterations").          SURVEY.md 8(a) a2-a4.
//
// Why generate code: in the generic kernel (kernels.cu, gate_block_kernel) tile bits, register bits, parameter slots,
// CNOT address maps and diagonal-segment structure are run-time data; two thirds of its instructions were address
// arithmetic and interpretation of that data.  Here they are literals: shared-memory offsets are immediates, every
// rotation is two packed FMAs per amplitude pair, a diagonal segment multiplies by tables whose shape is known.
#pragma once
#include <stdint.h>

#include <string>
#include <vector>

#include "hamiltonian.h"
#include "schedule.h"

namespace gv {

struct JitBlock {
    std::string name;          // extern "C" kernel name
    std::string source;        // complete translation unit
    uint32_t smem_bytes = 0;   // dynamic shared memory per thread block
    uint32_t threads = 0;      // threads per thread block
    int tiles_log2 = 0;        // log2(tiles per statevector) = n - k
    double fma_ops_per_amp = 0.0;   // FP lane operations (one FMA / MUL / ADD on one real) per amplitude and launch that the
                                    // schedule needs: 2 per rotation (tangent form), 4 per complex factor, 6 / 4 / 3 per pair
                                    // of a complex / real / imaginary W; what the ALU roofline in bench.py is counted in
};

// True when the generated kernels cover this program (tile and register sizes, stage counts, shared-memory budget).
bool jit_supported(const Program &p, int prec, std::string &why);

// Source of the kernel of block `bi`.  prec: 0 = complex64, 1 = complex128.
// occupancy: thread blocks per SM the kernel is compiled for (0 = default).
// staged_io: every tile goes through shared memory on both sides (otherwise the first / last stage of a block reads /
// writes global memory directly when it carries no CNOT run).
// interleave: thread blocks in groups of this many (a power of two) take neighbouring tiles at the same time (0, 1: off).
bool jit_generate(const Program &p, int bi, int prec, int occupancy, bool staged_io, int interleave, JitBlock &out, std::string &err);

// ---- expectation passes (jit_expect.cpp): one kernel per read-only pass of an ExpectPlan ------------------------------
struct JitExpectData {   // host images of the arrays the kernels read from global memory (uploaded once per Hamiltonian)
    struct Pat { uint32_t dst, begin, end, pad; };          // shared-memory byte offset of a table entry; its terms
    struct Term { double cr, ci; uint64_t zout, pad; };     // c_k i^{nY}; z bits outside the tile; (direct groups: local z mask)
    std::vector<double> wst;                                 // static W tables, (re, im) per entry, pass after pass
    std::vector<Pat> pats;
    std::vector<Term> terms;
    std::vector<uint32_t> pass_wst_off, pass_pat_off, pass_pat_cnt;   // per pass: first entry / first pattern / patterns
};
bool jit_expect_supported(const ExpectPlan &plan, int n, int prec, std::string &why);
// Appends pass `pi`'s arrays to `data` (call for pi = 0, 1, ... in order) and writes its kernel to `out`.
bool jit_expect_generate(const ExpectPlan &plan, int n, int prec, int pi, JitExpectData &data, JitBlock &out, std::string &err);

// ---- run time (jit_rt.cpp): NVRTC through dlopen, module load and launch through the driver entry points -----------
struct JitModule;   // one loaded kernel
bool jit_runtime_available(std::string &why);
// Compiles `blk.source` to an sm_100a image (cached per process by source text); needs no device.
bool jit_compile_only(const JitBlock &blk, std::vector<char> &cubin, std::string &err);
// Compiles (or takes the cached image) and loads it on the current device.
JitModule *jit_load(const JitBlock &blk, std::string &err);
void jit_unload(JitModule *m);
// Launch on `stream`: states (device), stride in amplitudes, ry / cs tables (device, per statevector row of P entries);
// per_cta: consecutive (statevector, tile) work items one thread block handles (its setup is paid once per thread block).
// src (optional): statevector(s) the tiles are read from instead of `states` (src_stride 0: all rows read the same one).
int jit_launch(JitModule *m, const JitBlock &blk, void *states, uint64_t stride, const void *ry, const void *cs, int nb, int P,
               int per_cta, void *stream, const void *src = nullptr, uint64_t src_stride = 0);
// Expectation pass: table = diagonal energy table, wst / pats = this pass's static tables and patterns, terms = all terms.
int jit_launch_expect(JitModule *m, const JitBlock &blk, const void *states, uint64_t stride, const void *table, const void *wst,
                      const void *pats, const void *terms, double *partial, uint32_t slots_per_b, uint32_t slot_off, int nb,
                      int per_cta, void *stream);

}  // namespace gv
