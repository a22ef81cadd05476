// afs_f32.cu -- the fp32 device entry points of include/afs.h (the product path)
#include "afs_run.cuh"

using namespace afs;

extern "C" afs_status afs_eval_grad(afs_problem* p, const float* X, int32_t B, float* F, float* G, void* stream)
{ return eval_grad_impl<float>(p, X, B, F, G, stream); }
extern "C" afs_status afs_round_count(afs_problem* p, const float* X, int32_t B, int8_t* assign, int32_t* sat, void* stream)
{ return round_count_impl<float>(p, X, B, assign, sat, stream); }
extern "C" afs_status afs_pgd_run(afs_problem* p, float* X, int32_t B, int32_t steps, float lr, const int8_t* mask,
                                  int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* stream)
{ return pgd_run_impl<float>(p, X, B, steps, lr, mask, best_assign, best_sat, best_step, stream); }

extern "C" afs_status afs_pgd_run_conv(afs_problem* p, float* X, int32_t B, int32_t max_steps, float lr, const int8_t* mask,
                                       float tol, int8_t* best_assign, int32_t* best_sat, int32_t* best_step,
                                       int32_t* conv_step, int32_t* final_sat, float* final_F, void* stream)
{ return pgd_run_conv_impl<float>(p, X, B, max_steps, lr, mask, tol, best_assign, best_sat, best_step, conv_step, final_sat, final_F, stream); }

extern "C" afs_status afs_pgd_run_masks(afs_problem* p, float* X, int32_t B, int32_t steps, float lr, const int8_t* masks,
                                        int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* stream)
{ return pgd_run_impl<float>(p, X, B, steps, lr, masks, best_assign, best_sat, best_step, stream, float(0), nullptr, true); }

extern "C" afs_status afs_constraint_grad_l1(afs_problem* p, const float* X, int32_t B, float* gm, void* stream)
{ return grad_l1_impl<float>(p, X, B, gm, stream); }
