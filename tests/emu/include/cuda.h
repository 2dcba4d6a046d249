// tests/emu: stands in for the CUDA driver header in the emulated TEST build (emu_cuda.h)
#pragma once
#include "../emu_cuda.h"
