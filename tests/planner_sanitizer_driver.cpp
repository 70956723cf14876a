// Driver of the -fsanitize=address,undefined build of the host planner (csrc/ppl_plan.cpp: plain C++, no CUDA call):
// ppl_plan_dry_ex over a grid of shapes x symmetry modes x workspace caps x debug knobs, the same entry point the planner
// tests call through ctypes.  Built and run by tests/test_planner_sanitizers_cpu.py; any sanitizer report aborts
// (-fno-sanitize-recover=all), so exit code 0 means a clean run.  SURVEY.md section 5 (race detection / sanitizers).
#include "../include/ppl.h"

#include <cstdio>
#include <cstring>

int main() {
    const int shapes[][3] = {{1, 1, 1},   {1, 2, 1},    {2, 3, 5},     {5, 20, 60},    {5, 53, 232},    {3, 37, 11},     {4, 35, 9},
                             {7, 131, 40}, {8, 56, 300}, {9, 57, 300},  {300, 16, 16},  {20, 200, 800},  {40, 190, 1150}, {40, 400, 1600}};
    // big shapes (Table 3 rows, xl, the former int overflow of step0_seconds at nvirt >= 2431): default knobs only
    const int big[][3] = {{60, 600, 2400}, {50, 950, 10000}, {100, 900, 5000}, {225, 575, 4000}, {2, 1000, 3}, {1, 2600, 2}};
    const size_t caps[] = {0, (size_t)64 << 20, (size_t)6 << 30};
    const size_t frees[] = {(size_t)178 << 30, (size_t)1 << 30};
    long ok = 0, refused = 0;
    auto one = [&](const int *s, int mode, size_t cap, size_t fr, int knob) -> int {
        ppl_debug_opts_t d;
        memset(&d, 0, sizeof(d));
        if (knob == 1) d.tile_edge = 8;
        if (knob == 2) d.ni_max = 3;
        if (knob == 3) d.full_tight = 1;
        if (knob == 4) d.full_tbg = 16, d.full_slots = 1;
        if (knob == 5) d.full_strips = 2, d.full_rect_tiles = 1;
        if (knob == 6) d.no_small_fused = 1, d.full_min_v = 2;
        if (knob == 7) d.cpasync_kernels = 1, d.full_no_diag_pack = 1;
        ppl_info_t info;
        memset(&info, 0, sizeof(info));
        const int rc = ppl_plan_dry_ex(s[0], s[1], s[2], cap, fr, knob == 2 ? 1 : 148, mode, knob ? &d : nullptr, &info);
        if (rc == PPL_OK) {
            ++ok;
            if (!(info.flops_executed >= info.flops_useful * 0.999) || info.n_tiles < 1) {
                printf("implausible plan for (%d,%d,%d) mode %d cap %zu knob %d\n", s[0], s[1], s[2], mode, cap, knob);
                return 2;
            }
        } else {
            ++refused;
        }
        return 0;
    };
    for (const auto &s : shapes)
        for (int mode = -1; mode <= PPL_SYM_FULL; ++mode)
            for (size_t cap : caps)
                for (size_t fr : frees)
                    for (int knob = 0; knob < 8; ++knob)
                        if (one(s, mode, cap, fr, knob)) return 2;
    for (const auto &s : big)
        for (int mode = -1; mode <= PPL_SYM_FULL; ++mode) {
            if (s[1] > 2000 && mode != 0) continue;  // (seconds per plan under ASan at this nvirt: once is enough)
            if (one(s, mode, 0, (size_t)178 << 30, 0)) return 2;
        }
    // argument errors must come back as codes
    ppl_info_t info;
    if (ppl_plan_dry(0, 5, 5, 0, (size_t)1 << 30, 148, -1, &info) != PPL_ERR_INVALID_ARG) return 3;
    if (ppl_plan_dry(5, 5, 5, 0, (size_t)1 << 30, 0, -1, &info) != PPL_ERR_INVALID_ARG) return 3;
    if (ppl_plan_dry(5, 5, 5, 0, (size_t)1 << 30, 148, 9, &info) != PPL_ERR_INVALID_ARG) return 3;
    if (ppl_plan_dry(5, 5, 5, 0, (size_t)1 << 30, 148, -1, nullptr) != PPL_ERR_INVALID_ARG) return 3;
    printf("planner under ASan + UBSan: %ld plans made, %ld requests refused, no report\n", ok, refused);
    return 0;
}
