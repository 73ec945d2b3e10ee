// ea_resident.cuh -- shared-memory-resident sweep kernel (L = 8, 16).  Filled in below.
#pragma once
#include "ea_device.cuh"
