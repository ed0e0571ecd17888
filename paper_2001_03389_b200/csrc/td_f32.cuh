// td_f32.cuh -- time-domain sigma cut for float32 (placeholder until the kernel lands)
#pragma once
#include "common.cuh"
