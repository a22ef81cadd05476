// afs_f64.cu -- the fp64 verification build of the same kernels (BASELINE.json north_star), *_f64 entry points
#include "afs_run.cuh"

using namespace afs;

extern "C" afs_status afs_eval_grad_f64(afs_problem* p, const double* X, int32_t B, double* F, double* G, void* stream)
{ return eval_grad_impl<double>(p, X, B, F, G, stream); }
extern "C" afs_status afs_round_count_f64(afs_problem* p, const double* X, int32_t B, int8_t* assign, int32_t* sat, void* stream)
{ return round_count_impl<double>(p, X, B, assign, sat, stream); }
extern "C" afs_status afs_pgd_run_f64(afs_problem* p, double* X, int32_t B, int32_t steps, double lr, const int8_t* mask,
                                      int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* stream)
{ return pgd_run_impl<double>(p, X, B, steps, lr, mask, best_assign, best_sat, best_step, stream); }

extern "C" afs_status afs_pgd_run_conv_f64(afs_problem* p, double* X, int32_t B, int32_t max_steps, double lr, const int8_t* mask,
                                       double tol, int8_t* best_assign, int32_t* best_sat, int32_t* best_step,
                                       int32_t* conv_step, int32_t* final_sat, double* final_F, void* stream)
{ return pgd_run_conv_impl<double>(p, X, B, max_steps, lr, mask, tol, best_assign, best_sat, best_step, conv_step, final_sat, final_F, stream); }

extern "C" afs_status afs_pgd_run_masks_f64(afs_problem* p, double* X, int32_t B, int32_t steps, double lr, const int8_t* masks,
                                        int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* stream)
{ return pgd_run_impl<double>(p, X, B, steps, lr, masks, best_assign, best_sat, best_step, stream, double(0), nullptr, true); }

extern "C" afs_status afs_constraint_grad_l1_f64(afs_problem* p, const double* X, int32_t B, double* gm, void* stream)
{ return grad_l1_impl<double>(p, X, B, gm, stream); }
