// Backward kernels (placeholder header; filled in by the backward milestone).
#pragma once
#include "sap_internal.h"
#include "sm100_ptx.cuh"
