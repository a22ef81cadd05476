// fp32 instantiation of the long-constraint launches
#include "afs_long_launch.cuh"
namespace afs {
template afs_status launch_long_all<float>(afs_problem*, const float*, const uint32_t*, const uint32_t*, int, float*, int32_t*, float*, const RunState*, cudaStream_t);
}
