// the runtime API, the execution model and the intrinsics all live in emu.h
#pragma once
#include "emu.h"
