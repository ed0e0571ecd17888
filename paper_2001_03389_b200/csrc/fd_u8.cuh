// fd_u8.cuh -- frequency-domain sigma cut (FDSC) for uint8 (placeholder until the kernel lands)
#pragma once
#include "common.cuh"
