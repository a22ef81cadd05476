// fp64 (verification build) instantiation of the long-constraint launches
#include "afs_long_launch.cuh"
namespace afs {
template afs_status launch_long_all<double>(afs_problem*, const double*, const uint32_t*, const uint32_t*, int, double*, int32_t*, double*, const RunState*, cudaStream_t);
}
