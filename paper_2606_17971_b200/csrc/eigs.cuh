// eigs.cuh -- S0: reference construction (filled in below).
#pragma once
#include "coarse.cuh"
