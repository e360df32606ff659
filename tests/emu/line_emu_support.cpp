// line_emu_support.cpp -- TEST ONLY: what the emulated launchers expect from the library besides their own file.
#include <cstdarg>
#include <cstdio>

#include "emu_rt.h"

namespace gspn {
static thread_local char g_err[2048] = "";
void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
}  // namespace gspn

extern "C" const char* emu_last_error() { return gspn::g_err; }
extern "C" void emu_set_jitter(int max_us, unsigned seed) { emu::jitter_us = max_us; emu::jitter_seed = seed ? seed : 1u; }
extern "C" void emu_set_lazy(int on) { emu::lazy = on != 0; }
