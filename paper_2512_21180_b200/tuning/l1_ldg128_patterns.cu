// microbenchmark: cost of LDG.128 gathers from L1 under controlled lane->address patterns
#include <cstdio>
#include <cuda_runtime.h>
#include <vector>
__global__ void k(const float4* __restrict__ buf, const int* __restrict__ pat, float* out, int iters, int stride_cells) {
    int lane = threadIdx.x & 31;
    int off = pat[lane];                       // cell offset for this lane
    const float4* p = buf + off;
    float acc = 0.f;
    int adv = 0;
    #pragma unroll 1
    for (int i = 0; i < iters; ++i) {
        #pragma unroll
        for (int j = 0; j < 8; ++j) {
            float4 v = __ldg(p + adv + j * stride_cells);
            acc += v.x + v.y + v.z + v.w;
        }
        adv = (adv + 8 * stride_cells) & 2047;   // stay inside a 32 KB window (+ pattern span)
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}
int main() {
    const int NC = 1 << 16;  // cells (1 MB) per buffer; all CTAs read the same window -> L1 hits
    float4* buf; cudaMalloc(&buf, NC * sizeof(float4)); cudaMemset(buf, 0, NC * sizeof(float4));
    int* dpat; cudaMalloc(&dpat, 32 * sizeof(int));
    float* out; cudaMalloc(&out, 148 * 8 * 256 * sizeof(float));
    struct P { const char* name; int pat[32]; };
    std::vector<P> pats;
    auto add = [&](const char* n, auto f) { P p; p.name = n; for (int l = 0; l < 32; ++l) p.pat[l] = f(l); pats.push_back(p); };
    // line = 8 cells. q = l/8 (quarter-warp), i = l%8
    add("A: qw reads 8 distinct cells of ONE line (coalesced)", [](int l) { return l; });
    add("B: all 32 lanes same cell (broadcast)", [](int l) { return 0; });
    add("C: qw = 8 lines, distinct bank groups (cell i of line i)", [](int l) { int q = l / 8, i = l % 8; return (q * 8 + i) * 8 + i; });
    add("D: qw = 8 lines, SAME bank group (cell 0 of each line)", [](int l) { int q = l / 8, i = l % 8; return (q * 8 + i) * 8; });
    add("E: qw = 2 lines x 4 cells, disjoint groups (0-3 | 4-7)", [](int l) { int q = l / 8, i = l % 8; return (q * 2 + i / 4) * 8 + i; });
    add("F: qw = 2 lines x 4 cells, same groups (0-3 | 0-3)", [](int l) { int q = l / 8, i = l % 8; return (q * 2 + i / 4) * 8 + (i % 4); });
    add("G: qw = 4 lines x 2 cells, disjoint groups", [](int l) { int q = l / 8, i = l % 8; return (q * 4 + i / 2) * 8 + i; });
    add("H: qw = 4 lines x 2 cells, same groups (0,1)", [](int l) { int q = l / 8, i = l % 8; return (q * 4 + i / 2) * 8 + (i % 2); });
    add("I: qw = 5 distinct cells in 3 lines w/ dups, disjoint groups", [](int l) { int q = l / 8, i = l % 8; int c[8] = {0, 0, 1, 1, 10, 10, 19, 20}; return q * 64 + c[i]; });
    add("J: qw = 3 distinct cells same line w/ dups", [](int l) { int q = l / 8, i = l % 8; int c[8] = {0, 0, 0, 1, 1, 1, 2, 2}; return q * 8 + c[i]; });
    add("K: pairs of lanes share a cell, 4 cells in one line", [](int l) { return (l / 8) * 8 + (l % 8) / 2; });
    add("L: 16 lanes/line: lanes 0-15 -> line0 cells (l%8), dup across qw", [](int l) { return (l / 16) * 8 + l % 8; });
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 4000;
    for (auto& p : pats) {
        cudaMemcpy(dpat, p.pat, sizeof(p.pat), cudaMemcpyHostToDevice);
        for (int stride : {8, 9}) {
            k<<<148 * 8, 256>>>(buf, dpat, out, 200, stride);
            cudaEventRecord(e0);
            k<<<148 * 8, 256>>>(buf, dpat, out, iters, stride);
            cudaEventRecord(e1); cudaEventSynchronize(e1);
            float ms; cudaEventElapsedTime(&ms, e0, e1);
            double req_per_sm = 8.0 * 8 * iters * 8;  // CTAs/SM * warps * iters * loads
            double cyc = ms * 1e-3 * 1.965e9;
            printf("%-62s stride %d: %.2f cycles per LDG.128 request per SM (%.3f ms)\n", p.name, stride, cyc / req_per_sm, ms);
        }
    }
    return 0;
}
