// lower.h -- Program (schedule.h) -> flat device arrays (devprog.h).  Pure host C++.
#pragma once
#include <string>
#include <vector>

#include "devprog.h"
#include "schedule.h"

namespace gv {

struct DevProgram {
    int n = 0, k = 0, f = 0, R = 0;
    std::vector<DBlock> blocks;
    std::vector<DStage> stages;
    std::vector<DOp> ops;
    std::vector<DSeg> segs;
    std::vector<DTrz> trzs;
    std::vector<uint64_t> tczs;
    std::vector<int32_t> csidx;   // block-local (cos,sin) slot -> parameter index
    std::vector<int16_t> ryl;     // RY layers: DEV_MAX_R block-local (cos,sin) slots each, -1 = no gate on the slot
    std::vector<DCx> cxs;         // trailing CNOT runs
    std::vector<uint32_t> slut;   // per-stage thread lookups (devprog.h SLUT_ENTRIES): 48 u32 then 48 u64 per stage
    uint32_t max_smem_prog = 0;   // largest per-block program slice (bytes)
};

// scs_bytes: sizeof one (cos,sin) pair in the working precision (8 for c64, 16 for c128).
bool lower_program(const Program &p, int scs_bytes, DevProgram &out, std::string &err);

// Bytes of the shared-memory program slice for given counts (layout used by the kernels, 16-byte aligned parts).
uint32_t prog_slice_bytes(uint32_t n_stages, uint32_t n_ops, uint32_t n_segs, uint32_t n_trz, uint32_t n_tcz,
                          uint32_t n_cs, uint32_t n_ryl, uint32_t n_cx, int scs_bytes);

}  // namespace gv
