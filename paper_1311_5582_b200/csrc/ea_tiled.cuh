// ea_tiled.cuh -- z-slab tiled sweep kernel (L = 32).  Filled in below.
#pragma once
#include "ea_device.cuh"
