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

#include "schedule.h"

namespace gv {

struct JitBlock {
    std::string name;          // extern "C" kernel name
    std::string source;        // complete translation unit
    uint32_t smem_bytes = 0;   // dynamic shared memory per thread block
    uint32_t threads = 0;      // threads per thread block
    int tiles_log2 = 0;        // log2(tiles per statevector) = n - k
};

// True when the generated kernels cover this program (tile and register sizes, stage counts, shared-memory budget).
bool jit_supported(const Program &p, int prec, std::string &why);

// Source of the kernel of block `bi`.  prec: 0 = complex64, 1 = complex128.
bool jit_generate(const Program &p, int bi, int prec, JitBlock &out, std::string &err);

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
int jit_launch(JitModule *m, const JitBlock &blk, void *states, uint64_t stride, const void *ry, const void *cs, int nb, int P,
               int per_cta, void *stream);

}  // namespace gv
