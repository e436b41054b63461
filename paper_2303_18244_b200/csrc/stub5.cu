#include "kernels.h"
namespace me {
static cudaError_t launch_stub(int, const LaunchArgs&) { return cudaErrorNotSupported; }
static const double cn[1] = {0};
extern const ProcTable tab_gg_ttxggg = {5, 1240, 0, 120, 324, 0, {0, 0, 0}, 0, cn, launch_stub, nullptr};
}
