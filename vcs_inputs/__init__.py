"""Seeded synthetic inputs (ROM images, env seeds, action streams) shared by the oracle tests and
the CUDA path's tests/bench.  Holds none of the emulator's arithmetic (task rule ③)."""
from .prng import SplitMix64, draws, env_seeds  # noqa: F401
from .asm6502 import Asm, hand_rom, OPCODES, TIA_W, TIA_R, RIOT  # noqa: F401
from .romgen import Features, FEATURES, make_rom  # noqa: F401
from .configs import Workload, make_workload  # noqa: F401
from .mapper_roms import superchip_rom, e0_rom, fe_rom  # noqa: F401
