// rod_adjoint.cuh — reverse pass (placeholder until the adjoint kernel lands)
#pragma once
#include "rod_substep.cuh"
