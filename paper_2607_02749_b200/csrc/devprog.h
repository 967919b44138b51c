// devprog.h -- device-side encoding of the compiled schedule and of the Hamiltonian passes.
// Plain PODs shared by the host lowering (lower.cpp, hamiltonian.cpp) and the kernels (kernels.cuh); the host
// builds arrays of these, uploads them into the caller's workspace, and every thread block copies the slice it
// needs into shared memory before it touches the state.                       SURVEY.md section 8(a) a0, a3-a7.
#pragma once
#include <stdint.h>

#include "program.h"

namespace gv {

constexpr int DEV_MAX_R = 5;
enum : uint8_t { MOP_RYL = 3 };   // device-only micro-op: RY on every register slot that has one (ryl[slot] >= 0)

// ---- gate engine ------------------------------------------------------------------------------------------
struct DOp {                 // 8 bytes; one register-level micro-op of a stage
    uint8_t kind;            // MOP_RYL (a layer of RY on distinct register slots) or MOP_DIAG
    uint8_t a;               // RY: register slot; CX: target slot
    uint8_t b;               // CX: control register slot (CTL_REG) or global qubit (CTL_FIXED)
    uint8_t c;               // CX: CTL_REG / CTL_FIXED
    int32_t idx;             // RYL: offset into the block's ryl array (DEV_MAX_R entries); DIAG: segment index
};

constexpr int TPH_CONST = 48;           // entry holding the product of the tile-constant RZ factors
constexpr int TPH_ENTRIES = 16 + 32 + 16;   // thread-phase tables of a segment: [0,16) over thread-index bits 0..3 (and all
                                       // tile-constant factors), [16,48) over thread-index bits 4..8
enum : uint8_t { TB_CONST = 254, TB_XREG = 200 };   // DTrz.tb: tile-constant qubit / TB_XREG + s: further RZ on slot s
enum : int { TCZ_LO = 0, TCZ_HI = 1, TCZ_CROSS = 2, TCZ_CLASS_SHIFT = 62 };   // class of a thread-level CZ pair

struct DTrz {                // RZ on a qubit that is not a register bit of the stage (thread- or tile-constant)
    uint8_t qubit;           // global qubit
    uint8_t tb;              // thread-index bit the qubit maps to in the segment's stage, TB_CONST, or TB_XREG + slot
    uint16_t cs;             // block-local (cos,sin) index
};

struct DSeg {                // one merged diagonal segment (all its RZ and CZ, Eq. 7 phases and CZ signs)
    uint16_t trz_begin, trz_end;        // DTrz entries (block-local); the TB_XREG entries come first
    uint16_t tcz_begin, tcz_end;        // CZ pairs with no register bit: two qubit bits + class in bits 62-63;
                                        // the TCZ_CROSS pairs come first
    int16_t reg_rz[DEV_MAX_R];          // per register slot: block-local (cos,sin) index of its RZ, or -1
    uint8_t stage;                      // block-local stage of the segment (fixes the thread-bit layout)
    uint8_t n_xreg;                     // TB_XREG entries
    uint32_t regreg_neg;                // bit r set: amplitude with register index r changes sign (reg-reg CZ)
    uint16_t n_cross;                   // TCZ_CROSS pairs
    uint16_t pad2;
    uint64_t nbr[DEV_MAX_R];            // per slot: global qubits CZ-coupled to it that are not register bits
};

constexpr int SLUT_ENTRIES = 16 + 32;   // per-stage thread lookup: [0,16) thread-index bits 0..3, [16,48) bits 4..8

struct DStage {              // 68 bytes
    uint8_t regbit[DEV_MAX_R];          // local bit position (inside the tile) of each register slot, ascending
    uint8_t has_cx;                     // the stage ends with a CNOT run
    uint16_t op_begin, op_end;          // DOp entries (block-local)
    uint16_t cx_begin, cx_end;          // DCx entries (block-local): the trailing CNOT run
    uint16_t postbit[DEV_MAX_R];        // image of the unit vector of each register bit under the CNOT run (linear part)
    uint8_t pad[2];
    uint32_t po_bytes[DEV_MAX_R];       // swizzled BYTE offset of each register bit: phys(1 << regbit) * sizeof(amplitude)
    uint32_t post_bytes[DEV_MAX_R];     // the same for postbit (write-back of a stage with a CNOT run)
};

struct DCx {                 // one CNOT of a trailing run, as an update of the LOCAL index: j ^= ctl_bit << tl
    uint8_t tl;              // target: local bit position
    uint8_t cl;              // control: local bit position, or 255 when the control qubit is outside the tile
    uint8_t cq;              // control: global qubit (used when cl == 255: bit of the tile base)
    uint8_t pad;
};

struct DBlock {              // one HBM round trip over every statevector in flight
    uint8_t k;               // tile bits
    uint8_t n_runs;
    uint8_t source_zero;     // 1: tile starts as |0...0> restricted to the tile (no global read)
    uint8_t n_stages;
    Run runs[MAX_RUNS];      // local bits [lpos,lpos+len) <-> global qubits [gpos,gpos+len)
    uint32_t stage_off, op_off, seg_off, trz_off, tcz_off, cs_off, ryl_off, cx_off;   // offsets into the device arrays
    uint32_t n_ops, n_segs, n_trz, n_tcz, n_cs, n_ryl, n_cx;
    uint32_t smem_prog_bytes;                                         // shared memory the slice needs (program + phase tables)
    uint32_t tph_off;                                                 // byte offset of the thread-phase tables in the slice
    uint32_t slut_off;       // byte offset of the per-stage thread lookups (SLUT_ENTRIES x (u32 + u64) per stage)
    uint32_t slut_goff;      // byte offset of their host-built image in the device slut array
    uint32_t off_tcz, off_segs, off_stages, off_ops, off_trz, off_cxs, off_ryl;   // byte offsets of the slice parts (cs = 0)
    uint32_t pad3;
    uint64_t hi[16];         // global offsets of the 16-byte vectors a thread moves: hi[i] = scatter(i * threads * V)
    uint32_t hip[16];        // their swizzled shared-memory element offsets: phys(i * threads * V)
    uint32_t lead_cx;        // 1: stage 0 is nothing but a CNOT run; it is applied while the tile is written to shared
                             // memory after the load (permuted addresses) and skipped in the stage loop
    uint32_t e1_cx;          // swizzled image of local index 1 under that run (second amplitude of a 16-byte vector)
    uint32_t hip_cx[16];     // swizzled images of i * threads * V under that run (linear part)
    uint32_t n_lead_cx;      // entries of lead_cxs (0 when the run is longer than the inline array: read from global)
    DCx lead_cxs[32];        // the leading CNOT run inline: as a kernel parameter it costs no global-load latency
    uint32_t n_cs_inline;    // entries of cs_inline (0: too many, read csidx from global)
    int32_t cs_inline[64];   // parameter index of each (cos,sin) slot, inline for the same reason (program + phase tables)
};

// ---- Hamiltonian engine -----------------------------------------------------------------------------------
struct DTerm {               // one Pauli term of an off-diagonal group, 32 bytes
    double cr, ci;           // c_k * i^{n_Y}
    uint64_t zout;           // z_mask bits outside the pass's tile bits (sign is constant per tile)
    uint32_t zu;             // z_mask bits inside the tile, compressed to the group's table index space
    uint32_t pad;
};

struct URun { uint8_t lpos, len, shift, pad; };   // table index bits: ((j >> lpos) & ((1<<len)-1)) << shift

struct DGroup {              // one flip mask (or a slice of its terms) inside a pass, 64 bytes
    uint32_t m_loc;          // flip mask in local tile coordinates (non-zero)
    uint32_t term_begin, term_end;
    uint32_t tab_off;        // offset of the group's W table in the shared-memory table area
    uint8_t ubits;           // table has 2^ubits entries (table mode)
    uint8_t n_uruns;
    uint8_t pivot;           // highest set bit of m_loc
    uint8_t direct;          // 1: no table; W is summed term by term per pair and DTerm.zu is the LOCAL z mask
    uint8_t last_in_batch;   // 1: tables of groups up to and including this one are built together
    uint8_t n_ex;            // table mode: entries of ex[] = 1 + loop bits
    uint8_t pad[2];
    uint32_t dyn_end;        // terms [term_begin, dyn_end) have z bits outside the tile (sign depends on the tile) and
                             // are added per thread block; terms [dyn_end, term_end) are folded into the static table
    uint32_t gtab_off;       // offset of the group's static W table in the global table array (= batch base + tab_off)
    uint32_t batch_entries;  // table entries of the whole batch this group belongs to
    uint32_t batch_last;     // index of the last group of that batch
    uint32_t uloc;           // table mode: the local bits that form the table index (ascending order = index bit order)
    uint64_t hot;            // what the group loop needs, one shared-memory read: mode (0 lookup, 1 register stage, 2 direct)
                             // | m_r << 2 | rs_id << 8 | tab_off << 24 | has tile-dependent terms << 63
    uint32_t ex_pack;        // ex[] packed 4 bits each (entry e at bits 4e)
    uint32_t lp_pack;        // lp[] packed 4 bits each
    uint64_t urun_pack;      // uruns packed 12 bits each: lpos | len << 4 | shift << 8
    uint8_t rs;              // 1: register-stage group: flip mask and table index live in the register bits of stage rs_id
    uint8_t m_r;             // its flip mask over the register slots
    uint16_t rs_id;          // index into the DRs array
    uint32_t pm_bytes;       // swizzled byte offset of the flip mask: phys(m_loc) * sizeof(amplitude)
    uint32_t gt_index;       // index of the group's lookup block (GT_WORDS uint32) in the group-table array
    URun uruns[3];
    uint8_t ex[8];           // ascending local bit positions that are NOT thread bits: the pivot and the loop bits
    uint8_t lp[8];           // the loop bits (n_ex - 1 of them): local positions outside the table index bits, so
                             // that W is constant over a thread's pairs
};

// Per-group lookup block (host-built, tile-independent), GT_WORDS uint32:
//   [0,16)  low table : thread-index bits 0..3 -> swizzled byte offset of the thread's local index | table index << 20
//   [16,32) high table: thread-index bits 4..  -> same; the thread's word is low ^ high (both maps are GF(2)-linear)
//   [32,64) swizzled byte offsets of the 2^L loop-bit combinations
constexpr int GT_WORDS = 64;
constexpr int GT_BATCH_MAX = 32;   // groups per table batch (shared-memory copy of their lookup blocks)

// Register stage of the expectation kernel: every thread holds the 2^R amplitudes that differ in these local bits; all
// groups whose flip mask and z bits lie inside them are evaluated from registers (partner = another register).
struct DRs {
    uint8_t regbit[DEV_MAX_R];     // local bit positions, ascending
    uint8_t pad[3];
    uint32_t po_bytes[DEV_MAX_R];  // swizzled byte offset of each register bit
};

struct DPass {               // one read-only sweep over the state
    uint8_t k, n_runs, with_diag, pad;
    Run runs[MAX_RUNS];
    uint32_t group_begin, group_end;
    uint32_t n_batches;      // <= PASS_MAX_BATCHES (longer passes are cut into several with the same tile bits)
    uint32_t pad2;
    uint64_t hi[64];         // as DBlock::hi for the expectation kernel's thread count
    struct Batch { uint32_t g_first, g_last, entries, wbase; } batch[12];   // groups [g_first, g_last], their table entries,
                                                                            // offset of their static tables in the wstat array
};
constexpr int PASS_MAX_BATCHES = 12;

}  // namespace gv
