// pf_krylov_tiled.cu -- placeholder until the tiled kernels land: reports "unsupported" so that
// the driver uses the direct family.
#include "pf_launch.h"
namespace pf {
bool tiled_supported(const GridDims&) { return false; }
void launch_residual_tiled(const LaunchCtx&, const Operator&, const KrylovVecs&, int) {}
void launch_k1_tiled(const LaunchCtx&, const Operator&, const KrylovVecs&, bool) {}
void launch_k2_tiled(const LaunchCtx&, const Operator&, const KrylovVecs&, bool) {}
}
