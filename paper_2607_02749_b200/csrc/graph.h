// graph.h -- host side of Graph-VQE's Hamiltonian-aware partitioning (north_star item 3):
// weighted qubit interaction graph (Eq. 9), modularity (Eq. 10), Louvain
// community detection and the merge of blocks below S_min.  Pure host C++, no GPU work.
#pragma once
#include <stdint.h>

#include <vector>

namespace gv {

// Dense symmetric weight matrix, row-major n x n, zero diagonal unless the caller supplies self loops.
// Q of Eq. 10 with resolution gamma (gamma = 1 is the paper's formula); 0 when the graph has no weight.
double modularity(int n, const double *w, const int32_t *community, double gamma);

// Louvain (local moving in ascending node order + aggregation, repeated until a level moves nothing).
// community[i] in [0, K): labels in order of first appearance by ascending node.  Returns K.
int louvain(int n, const double *w, double gamma, int32_t *community);

// Blocks with fewer than s_min nodes are merged, smallest first, into the block they share the most weight with.
// Labels are renumbered by first appearance.  Returns the new K.
int merge_small_blocks(int n, const double *w, int s_min, int32_t *community);

// Renumber labels by first appearance (ascending node); returns K.
int relabel_first_appearance(int n, int32_t *community);

}  // namespace gv
