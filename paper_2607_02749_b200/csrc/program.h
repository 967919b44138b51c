// program.h -- compiled schedule ("program") shared by the host compiler (schedule.cpp) and the kernels.
// Plain PODs only; the same bytes are interpreted on the host and uploaded to the device workspace.
//
// A *block* is one HBM round trip over all statevectors: a tile = the 2^k amplitudes whose index differs only
// in the block's tile bits T (k qubits, lowest f of them always qubits 0..f-1 so that every global access is a
// run of >= 2^f contiguous amplitudes).  Inside a block the tile lives in shared memory and is processed in
// *stages*: in a stage every thread owns the 2^R amplitudes that differ in the stage's R register bits and
// applies the stage's micro-ops in registers.  Diagonal gates (RZ, CZ) are merged into *diagonal segments*
// (one complex multiply per amplitude per segment).           SURVEY.md section 8(a) rows a0, a3, a4.
#pragma once
#include <stdint.h>

namespace gv {

enum : uint8_t { MOP_RY = 0, MOP_CX = 1, MOP_DIAG = 2 };
enum : uint8_t { CTL_REG = 0, CTL_FIXED = 1 };

struct MicroOp {      // 8 bytes
    uint8_t kind;     // MOP_*
    uint8_t a;        // RY: register slot; CX: target slot
    uint8_t b;        // CX: control = register slot (CTL_REG) or global qubit (CTL_FIXED)
    uint8_t c;        // CX: CTL_*
    int32_t param;    // RY: parameter index; DIAG: diagonal segment index (global numbering)
};

struct DiagRZ {       // e^{-i phi/2} on bit 0, e^{+i phi/2} on bit 1   (Eq. 7)
    uint8_t qubit;    // global qubit
    uint8_t slot;     // register slot of the owning stage, 255 = not a register bit
    uint16_t pad;
    int32_t param;
};

struct DiagCZ {       // sign -1 when both bits are set
    uint8_t q0, q1;   // global qubits
    uint8_t s0, s1;   // register slots or 255
};

struct DiagSeg {      // 16 bytes
    uint32_t rz_begin, rz_end;  // into the DiagRZ array
    uint32_t cz_begin, cz_end;  // into the DiagCZ array
};

constexpr int MAX_R = 5;
constexpr int MAX_RUNS = 8;

struct Stage {        // 32 bytes
    uint8_t regbit[MAX_R];      // LOCAL bit position (0..k-1) of each register slot, ascending
    uint8_t regq[MAX_R];        // the global qubit of each slot
    uint8_t n_seg;              // diagonal segments used by this stage
    uint8_t pad;
    uint32_t op_begin, op_end;  // into the MicroOp array
    uint32_t seg_begin;         // first diagonal segment of this stage (its R-tables are built per stage)
    uint32_t cx_begin, cx_end;  // trailing CNOT run of the stage (into the StageCx array): applied as an index
                                // permutation when the stage writes its amplitudes back (no register work)
};

struct StageCx { uint8_t tq, cq; };   // CNOT: target qubit, control qubit (global numbering)

// T as runs of consecutive qubits: local bits [lpos, lpos+len) <-> global qubits [gpos, gpos+len)
struct Run { uint8_t lpos, gpos, len, pad; };

struct Block {        // 64 bytes header
    uint8_t k;                  // tile bits
    uint8_t n_runs;
    uint8_t source_zero;        // 1: the tile is |0...0> (no read), SURVEY a2
    uint8_t pad;
    uint32_t stage_begin, stage_end;   // into the Stage array
    uint32_t max_seg;                  // max diagonal segments in one stage (R-table shared memory)
    Run runs[MAX_RUNS];
    uint32_t pad2[4];
};

}  // namespace gv
