#include "route_launch.cuh"
namespace gimbal {
GIMBAL_DEFINE_E(16)
}
