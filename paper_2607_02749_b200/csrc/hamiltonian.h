// hamiltonian.h -- host side of the Hamiltonian engine: Pauli strings -> integer masks
// -> canonical flip-mask groups ("Hamiltonian batching", PAPER.md:214-219 / Eq. 12, re-read as grouping by the
// X/Y flip mask) -> read-only passes over the state.  Pure host C++.
#pragma once
#include <stdint.h>

#include <string>
#include <vector>

#include "devprog.h"

namespace gv {

struct HostTerm { uint64_t x, z; int ny; double c; };

struct Hamiltonian {
    int n = 0;
    std::vector<HostTerm> terms;            // input order
    std::vector<int32_t> group_of_term;     // rank of the term's x mask among the distinct masks, ascending
    std::vector<uint64_t> group_mask;       // distinct x masks, ascending unsigned order (0 first when present)
    std::vector<uint64_t> diag_z;           // distinct z masks of the Z-only terms, ascending
    std::vector<double> diag_c;             // their coefficients summed in input order
    double abs_sum = 0.0;
};

// P|x> = i^{nY} (-1)^{popcount(x & z)} |x ^ xmask>  with x = X|Y positions, z = Z|Y positions   (Eq. 6)
bool hamiltonian_from_paulis(int n, int M, const char *paulis, const double *coeffs, Hamiltonian &H, std::string &err);
bool hamiltonian_from_masks(int n, int M, const uint64_t *xm, const uint64_t *zm, const double *coeffs, Hamiltonian &H,
                            std::string &err);

struct ExpectPlan {
    int k = 0;
    std::vector<DPass> passes;
    std::vector<DGroup> groups;
    std::vector<DTerm> terms;
    std::vector<DRs> rss;        // register stages
    std::vector<uint32_t> gtabs; // GT_WORDS words per table-mode group (see devprog.h)
    std::vector<double> wstat;   // static W tables (re, im interleaved), laid out batch by batch like the smem area
};

// n_store: qubits of the stored state; k/f: tile bits / fixed low tile bits; umax: largest table (bits);
// tab_cap: complex entries of the shared-memory table area.
// amp_bytes: 8 (complex64) or 16 (complex128): fixes the shared-memory swizzle and the byte offsets of the lookups.
// register_stages: evaluate the groups that fit R local bits from registers (false: every group takes the lookup / direct path).
bool plan_expectation(const Hamiltonian &H, int n_store, int k, int f, int umax, uint32_t tab_cap, int amp_bytes,
                      bool register_stages, ExpectPlan &plan, std::string &err);

}  // namespace gv
