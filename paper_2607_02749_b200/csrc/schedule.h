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
// from_zero: the first block starts from |0...0> without reading (false when a product-state prefix wrote the state).
// mid_cx: CNOTs whose target is a register qubit of the stage are applied in registers (MOP_CX micro-ops) and rotations
// may follow them in the same stage -- fewer stages on CNOT ansaetze; only the specialised kernels (jit.cpp) run such
// programs, the generic kernel needs mid_cx = false (every CNOT in a trailing run).
bool compile_program(int n, const std::vector<HostOp> &ops, int k, int f, int R, Program &out, std::string &err,
                     bool from_zero = true, bool mid_cx = false);

// Product-state prefix: the leading run of single-qubit rotations followed by the run of entanglers
// that comes before the next rotation.  RZ RY |0> on every qubit is a product state, CZ multiplies it by a sign, a
// CNOT permutes indices, so  psi[y] = sign(y) * prod_q f_q[(A^-1 y)_q]  can be WRITTEN without reading anything.
struct Prefix {
    int n_ops = 0;                         // ops [0, n_ops) of the list are covered (0 = no prefix)
    std::vector<int32_t> rot_begin;        // per qubit: range into rot_kind / rot_param (n + 1 entries)
    std::vector<uint8_t> rot_kind;         // 0 RY, 1 RZ, in application order
    std::vector<int32_t> rot_param;
    std::vector<uint8_t> cx_t, cx_c;       // CNOTs in list order (target, control); empty when the run is CZ
    int n_cz = 0;                          // CZ run as sum over distances d: popcount(y & (y >> d) & mask_d)
    int cz_d[4] = {0, 0, 0, 0};
    uint64_t cz_m[4] = {0, 0, 0, 0};
};
Prefix find_prefix(int n, const std::vector<HostOp> &ops);

std::string dump_program(const Program &p);

}  // namespace gv
