// graph.cpp -- interaction-graph partitioning for Graph-VQE (see graph.h).  Dense matrices: n is a qubit count.
#include "graph.h"

#include <algorithm>

namespace gv {

namespace {
constexpr double GAIN_EPS = 1e-12;   // a move must beat staying by more than this (reading G2)
}

int relabel_first_appearance(int n, int32_t *community)
{
    std::vector<int32_t> map;
    int32_t maxl = -1;
    for (int i = 0; i < n; ++i) maxl = std::max(maxl, community[i]);
    map.assign((size_t)maxl + 1, -1);
    int K = 0;
    for (int i = 0; i < n; ++i) {
        int32_t &m = map[(size_t)community[i]];
        if (m < 0) m = K++;
        community[i] = m;
    }
    return K;
}

// Eq. 10: Q = 1/(2m) sum_ij [w_ij - gamma k_i k_j / (2m)] delta(c_i, c_j), 2m = sum_ij w_ij.
double modularity(int n, const double *w, const int32_t *community, double gamma)
{
    std::vector<double> k((size_t)n, 0.0);
    double two_m = 0.0;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) { k[i] += w[(size_t)i * n + j]; two_m += w[(size_t)i * n + j]; }
    if (!(two_m > 0.0)) return 0.0;
    double q = 0.0;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j)
            if (community[i] == community[j]) q += w[(size_t)i * n + j] - gamma * k[i] * k[j] / two_m;
    return q / two_m;
}

// One level of local moving on the (super-)graph a (m x m, self loops on the diagonal).  Returns true if any
// node moved; comm receives labels by first appearance.
static bool local_moving(int m, const std::vector<double> &a, double gamma, double two_m, std::vector<int32_t> &comm)
{
    std::vector<double> k((size_t)m, 0.0), tot((size_t)m, 0.0), to_comm((size_t)m);
    for (int i = 0; i < m; ++i) for (int j = 0; j < m; ++j) k[i] += a[(size_t)i * m + j];
    comm.resize((size_t)m);
    for (int i = 0; i < m; ++i) { comm[i] = i; tot[i] = k[i]; }
    bool any = false, moved = true;
    while (moved) {
        moved = false;
        for (int i = 0; i < m; ++i) {
            const int32_t home = comm[i];
            std::fill(to_comm.begin(), to_comm.end(), 0.0);
            for (int j = 0; j < m; ++j) if (j != i) to_comm[(size_t)comm[j]] += a[(size_t)i * m + j];
            tot[(size_t)home] -= k[i];   // i taken out of its community
            // gain of joining community c, up to the common factor 1/m:  k_{i,in}(c) - gamma * tot(c) * k_i / (2m)
            const double stay = to_comm[(size_t)home] - gamma * tot[(size_t)home] * k[i] / two_m;
            double best = stay;
            int32_t best_c = home;
            for (int32_t c = 0; c < m; ++c) {   // ascending labels: ties go to the lowest label, staying wins ties
                if (c == home || !(to_comm[(size_t)c] > 0.0)) continue;
                const double g = to_comm[(size_t)c] - gamma * tot[(size_t)c] * k[i] / two_m;
                if (g > best + GAIN_EPS) { best = g; best_c = c; }
            }
            tot[(size_t)best_c] += k[i];
            if (best_c != home) { comm[i] = best_c; moved = true; any = true; }
        }
    }
    relabel_first_appearance(m, comm.data());
    return any;
}

int louvain(int n, const double *w, double gamma, int32_t *community)
{
    for (int i = 0; i < n; ++i) community[i] = i;
    if (n <= 0) return 0;
    double two_m = 0.0;
    for (size_t t = 0; t < (size_t)n * n; ++t) two_m += w[t];
    if (!(two_m > 0.0)) return n;   // no edges: every qubit is its own block
    int m = n;
    std::vector<double> a(w, w + (size_t)n * n);
    std::vector<int32_t> comm;
    while (true) {
        if (!local_moving(m, a, gamma, two_m, comm)) break;
        int K = 0;
        for (int i = 0; i < m; ++i) K = std::max(K, comm[i] + 1);
        for (int i = 0; i < n; ++i) community[i] = comm[(size_t)community[i]];
        // aggregation: A'_CD = sum_{i in C, j in D} A_ij (so 2m and the degrees are preserved)
        std::vector<double> b((size_t)K * K, 0.0);
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < m; ++j) b[(size_t)comm[i] * K + comm[j]] += a[(size_t)i * m + j];
        a.swap(b);
        m = K;
    }
    return relabel_first_appearance(n, community);
}

int merge_small_blocks(int n, const double *w, int s_min, int32_t *community)
{
    int K = relabel_first_appearance(n, community);
    while (K > 1) {
        std::vector<int> size((size_t)K, 0);
        for (int i = 0; i < n; ++i) ++size[(size_t)community[i]];
        int small = -1;
        for (int c = 0; c < K; ++c)
            if (size[c] < s_min && (small < 0 || size[c] < size[small])) small = c;   // smallest, then lowest label
        if (small < 0) break;
        std::vector<double> link((size_t)K, 0.0);
        for (int i = 0; i < n; ++i)
            if (community[i] == small)
                for (int j = 0; j < n; ++j)
                    if (community[j] != small) link[(size_t)community[j]] += w[(size_t)i * n + j];
        int target = -1;
        for (int c = 0; c < K; ++c)
            if (c != small && (target < 0 || link[c] > link[target])) target = c;    // largest weight, then lowest label
        for (int i = 0; i < n; ++i) if (community[i] == small) community[i] = target;
        K = relabel_first_appearance(n, community);
    }
    return K;
}

}  // namespace gv
