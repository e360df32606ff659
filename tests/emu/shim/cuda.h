// Shim of <cuda.h> for tests/emu (TEST ONLY): the tensor map is 128 opaque bytes; emu_ptx.h keeps its own record inside.
#pragma once
#include <cstdint>
struct alignas(64) CUtensorMap { uint64_t opaque[16]; };
