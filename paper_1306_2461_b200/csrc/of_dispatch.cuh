// of_dispatch.cuh -- radius dispatch (a run-time window radius selects a template instantiation) and the entry points of the
// other translation units.  The hoisted (of_set_hoist) instantiations of the persistent solve kernel are compiled in
// optflow_hoist.cu and the masked (of_set_mask) instantiations of K2, K3 and the solve kernel in optflow_mask.cu, in parallel with
// optflow.cu: together they are two thirds of the build time and share nothing but headers with the rest.
#pragma once
#include "of_solve.cuh"

#define DISPATCH_R(R_, CALL)                                                                       \
    switch (R_) {                                                                                  \
    case 1: { constexpr int R = 1; CALL; } break;   case 2: { constexpr int R = 2; CALL; } break;   \
    case 3: { constexpr int R = 3; CALL; } break;   case 4: { constexpr int R = 4; CALL; } break;   \
    case 5: { constexpr int R = 5; CALL; } break;   case 6: { constexpr int R = 6; CALL; } break;   \
    case 7: { constexpr int R = 7; CALL; } break;   case 8: { constexpr int R = 8; CALL; } break;   \
    case 9: { constexpr int R = 9; CALL; } break;   case 10: { constexpr int R = 10; CALL; } break; \
    case 11: { constexpr int R = 11; CALL; } break; case 12: { constexpr int R = 12; CALL; } break; \
    case 13: { constexpr int R = 13; CALL; } break; case 14: { constexpr int R = 14; CALL; } break; \
    case 15: { constexpr int R = 15; CALL; } break; case 16: { constexpr int R = 16; CALL; } break; \
    default: break;                                                                                \
    }

// Radius and window form: CALL sees `constexpr int R` and `constexpr bool BX` (BX only for box windows of radius >= 4, of_common.cuh).
#define DISPATCH_RB_CASE(N, BOX_, CALL)                                                            \
    case N: { constexpr int R = N;                                                                 \
              if ((BOX_) && win_box_path(N)) { constexpr bool BX = win_box_path(N); CALL; }        \
              else { constexpr bool BX = false; CALL; } } break;
#define DISPATCH_RB(R_, BOX_, CALL)                                                                \
    switch (R_) {                                                                                  \
    DISPATCH_RB_CASE(1, BOX_, CALL) DISPATCH_RB_CASE(2, BOX_, CALL) DISPATCH_RB_CASE(3, BOX_, CALL) DISPATCH_RB_CASE(4, BOX_, CALL)     \
    DISPATCH_RB_CASE(5, BOX_, CALL) DISPATCH_RB_CASE(6, BOX_, CALL) DISPATCH_RB_CASE(7, BOX_, CALL) DISPATCH_RB_CASE(8, BOX_, CALL)     \
    DISPATCH_RB_CASE(9, BOX_, CALL) DISPATCH_RB_CASE(10, BOX_, CALL) DISPATCH_RB_CASE(11, BOX_, CALL) DISPATCH_RB_CASE(12, BOX_, CALL)  \
    DISPATCH_RB_CASE(13, BOX_, CALL) DISPATCH_RB_CASE(14, BOX_, CALL) DISPATCH_RB_CASE(15, BOX_, CALL) DISPATCH_RB_CASE(16, BOX_, CALL) \
    default: break;                                                                                \
    }

// optflow_hoist.cu: of_solve_pair<R, false, true>; forwards to optflow_hoist_mask.cu (of_solve_pair<R, true, true>) when mk is set.
// Launch (cooperative, `sms` CTAs) and one-time attribute set-up (both units).
cudaError_t of_launch_solve_hoisted(int R, bool mk, const SolveArgs &a, int sms, cudaStream_t st);
cudaError_t of_setup_attrs_hoisted(int R, int smem_max);
cudaError_t of_launch_solve_hoisted_masked(int R, const SolveArgs &a, int sms, cudaStream_t st);
cudaError_t of_setup_attrs_hoisted_masked(int R, int smem_max);

// optflow_mask.cu: k2_products_hsum<R, true>, k3_vsum_solve<R, true>, of_solve_pair<R, true, false>.
void of_launch_k2_masked(int R, const K2Params &p, int grid, int threads, size_t smem, cudaStream_t st);
void of_launch_k3_masked(int R, const CUtensorMap &tm, const K3Params &p, int grid, int threads, size_t smem, cudaStream_t st);
cudaError_t of_launch_solve_masked(int R, const SolveArgs &a, int sms, cudaStream_t st);
cudaError_t of_setup_attrs_masked(int R, int smem_max);

// optflow_dual.cu: of_solve_dual<R, BX> (of_solve_dual.cuh), two pairs of two handles in one cooperative launch (unmasked, un-hoisted).
cudaError_t of_launch_solve_dual(int R, const SolveArgs &a0, const SolveArgs &a1, int sms, cudaStream_t st);
cudaError_t of_setup_attrs_dual(int R, int smem_max);
