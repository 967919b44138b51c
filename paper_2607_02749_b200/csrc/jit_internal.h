// jit_internal.h -- helpers shared by the two kernel generators (jit.cpp: gate blocks, jit_expect.cpp: expectation passes).
#pragma once
#include <stdint.h>

#include <cstdarg>
#include <cstdio>
#include <string>

namespace gv {
namespace {

struct Emit {
    std::string s;
    void operator()(const char *fmt, ...)
    {
        char buf[1024];
        va_list ap, ap2;
        va_start(ap, fmt);
        va_copy(ap2, ap);
        const int need = vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        if (need >= (int)sizeof buf) {   // long lines (constant arrays)
            std::string big((size_t)need + 1, ' ');
            vsnprintf(&big[0], big.size(), fmt, ap2);
            big.resize((size_t)need);
            s += big;
        } else s += buf;
        va_end(ap2);
        s += '\n';
    }
};

struct Geo {
    int k, R, TB, lv, prec;   // lv: log2(amplitudes per 16-byte unit)
    uint32_t pu(uint32_t u) const { return u ^ ((u >> 3) & 7u) ^ ((u >> 6) & 7u) ^ ((u >> 9) & 7u); }
    uint32_t off(uint32_t j) const { return (pu(j >> lv) << 4) | ((j & ((1u << lv) - 1u)) << 3); }
};


// Device-side prelude common to both generators: types, complex helpers, cp.async, the shared-memory offset function.
inline void emit_common_prelude(Emit &E, int prec, int lv)
{
    const char *T = prec == 0 ? "float" : "double";
    E("typedef %s real;", T);
    E("typedef %s2 amp;", T);
    E("typedef unsigned long long u64;");
    if (prec == 0) E("#define MK(x, y) make_float2((x), (y))");
    else E("#define MK(x, y) make_double2((x), (y))");
    E("struct __align__(16) unit16 { unsigned x, y, z, w; };");
    E("__device__ __forceinline__ void cp16(void *dst, const void *src) {");
    E("    asm volatile(\"cp.async.cg.shared.global [%%0], [%%1], 16;\" :: \"r\"((unsigned)__cvta_generic_to_shared(dst)), \"l\"(src));");
    E("}");
    E("__device__ __forceinline__ void cp_wait() { asm volatile(\"cp.async.wait_all;\" ::: \"memory\"); }");
    E("__device__ __forceinline__ unsigned OFF(unsigned j) { const unsigned u = j >> %d; return ((u ^ ((u >> 3) & 7u) ^ ((u >> 6) & 7u) ^ ((u >> 9) & 7u)) << 4) | ((j & %uu) << 3); }",
      lv, (1u << lv) - 1u);
}

// thread-index bit -> local bit for a phase whose "register" bits are regbits[0..nreg): the lanes of one shared-memory
// wavefront get local bits whose unit positions differ modulo 3 (conflict free under the fold of Geo::pu)
inline void choose_thread_bits_for(const Geo &g, const uint8_t *regbits, int nreg, int *tb)
{
    bool isreg[16] = {false};
    for (int s = 0; s < nreg; ++s) isreg[regbits[s]] = true;
    bool used[16] = {false};
    int n = 0;
    if (g.lv == 1 && !isreg[0]) { tb[n++] = 0; used[0] = true; }   // 8-byte accesses: the amplitude inside the unit varies fastest
    for (int res = 0; res < 3; ++res)
        for (int b = g.lv; b < g.k; ++b)
            if (!isreg[b] && !used[b] && (b - g.lv) % 3 == res) { tb[n++] = b; used[b] = true; break; }
    for (int b = 0; b < g.k; ++b) if (!isreg[b] && !used[b]) { tb[n++] = b; used[b] = true; }
}

// emits "unsigned NAME = deposit of tid bits into local bits tb[]"
inline void emit_deposit(Emit &E, const char *indent, const char *name, const int *tb, int TB)
{
    E("%sunsigned %s = 0u;", indent, name);
    for (int i = 0; i < TB;) {
        int len = 1;
        while (i + len < TB && tb[i + len] == tb[i] + len) ++len;
        E("%s%s |= ((tid >> %d) & %uu) << %d;", indent, name, i, (1u << len) - 1u, tb[i]);
        i += len;
    }
}

}  // namespace
}  // namespace gv
