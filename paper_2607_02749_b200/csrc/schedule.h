// schedule.h -- host-side schedule compiler: op list -> fused blocks -> register stages (
// PAPER.md:179 "compiled once and reused across all optimization iterations").  Pure host C++, no CUDA.
#pragma once
#include <stdint.h>

#include <string>
#include <vector>

#include "program.h"

namespace gv {

struct HostOp { int kind, q0, q1, param; };  // kinds = gvqe_opkind: 0 RY, 1 RZ, 2 CZ, 3 CNOT(target q0, control q1)

struct Program {
    int n = 0;        // qubits of the stored state (>= user n: small problems are padded with idle qubits)
    int k = 0;        // tile bits per block (<= n)
    int f = 0;        // fixed low tile bits
    int R = 0;        // register bits per stage
    std::vector<Block> blocks;
    std::vector<Stage> stages;
    std::vector<MicroOp> mops;
    std::vector<DiagSeg> segs;
    std::vector<DiagRZ> rzs;
    std::vector<DiagCZ> czs;
    std::vector<StageCx> cxs;
    // bookkeeping for tests: for every block the ops (indices into the input list) in execution order
    std::vector<std::vector<int>> block_ops;
    // every input op exactly once, in the order the device executes them (stages flattened, segments expanded)
    std::vector<int> exec_order;
};

// Compile.  Returns false and sets err on failure (never throws).
bool compile_program(int n, const std::vector<HostOp> &ops, int k, int f, int R, Program &out, std::string &err);

std::string dump_program(const Program &p);

}  // namespace gv
