"""ctypes loader for the CPU oracle (oracle/ovcs.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_DIR, "libovcs.so")
_SRC = [os.path.join(_DIR, f) for f in ("ovcs.c", "ovcs.h", "ovcs_cpu.inc", "ovcs_api.inc", "ovcs_soft.inc")]


def build(force: bool = False) -> str:
    """gcc -O2 the oracle into oracle/libovcs.so (rebuilt when a source is newer)."""
    stale = force or not os.path.exists(_SO) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if stale:
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-Wall", "-shared", "-fPIC", "-o", tmp, _SRC[0], "-lm"], cwd=_DIR)
        os.replace(tmp, _SO)
    return _SO


class Rom(C.Structure):
    _fields_ = [("data", C.POINTER(C.c_uint8)), ("size", C.c_uint32), ("mapper", C.c_uint32)]


MAPPERS = {"": 0, "2K": 1, "4K": 2, "F8": 3, "F6": 4, "F4": 5, "F8SC": 6, "F6SC": 7, "F4SC": 8, "E0": 9, "FE": 10}   # OVCS_MAP_*


class Config(C.Structure):
    _fields_ = [("y0", C.c_int32), ("max_lines", C.c_int32), ("f8_start_bank", C.c_int32), ("flags", C.c_uint32)]


REGS_DTYPE = np.dtype([("cycles", "<u8"), ("frame", "<u4"), ("pc", "<u2"), ("a", "u1"), ("x", "u1"), ("y", "u1"),
                       ("sp", "u1"), ("p", "u1"), ("bank", "u1"), ("line", "<u2"), ("cyc_in_line", "u1"),
                       ("status", "u1"), ("intim", "u1"), ("timint", "u1"), ("pad", "u1", (6,))])
assert REGS_DTYPE.itemsize == 32


class Debug(C.Structure):
    _fields_ = [(n, C.c_uint8) for n in ("posP0", "posP1", "posM0", "posM1", "posBL", "fresh", "hmove_blank", "vsync",
                                         "vblank", "latch_en", "wsync", "inpt4_latch", "grp0_new", "grp0_old",
                                         "grp1_new", "grp1_old")] + \
               [("cx", C.c_uint16), ("timer", C.c_uint8), ("tflag", C.c_uint8), ("shift", C.c_uint8),
                ("sub", C.c_uint16), ("clocks_rendered", C.c_uint64), ("n_instr", C.c_uint64), ("n_tia_writes", C.c_uint64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        P = C.c_void_p
        L.ovcs_create.argtypes = [C.POINTER(P), C.c_int32, C.POINTER(Rom), C.c_int32, P, P, C.POINTER(Config)]
        L.ovcs_reset.argtypes = [P, P]
        L.ovcs_step.argtypes = [P, P, C.c_int32]
        L.ovcs_step_masked.argtypes = [P, P, C.c_int32, P]
        L.ovcs_step_masked_range.argtypes = [P, P, C.c_int32, P, C.c_int32, C.c_int32]
        L.ovcs_set_switches.argtypes = [P, P]
        L.ovcs_boot.argtypes = [P, P, C.c_int32, C.c_int32, P, C.c_int32, C.c_int32]
        L.ovcs_step_range.argtypes = [P, P, C.c_int32, C.c_int32, C.c_int32]
        L.ovcs_step_instructions_range.argtypes = [P, P, C.c_int32, C.c_int32, C.c_int32]
        L.ovcs_step_instructions_soft_range.argtypes = [P, P, C.c_int32, C.c_double, C.c_double, C.c_int32, P, C.c_int32, C.c_int32]
        L.ovcs_detect_mapper.argtypes = [P, C.c_uint32]
        for f in ("ovcs_get_ram", "ovcs_get_regs", "ovcs_get_screen", "ovcs_get_cart_ram"):
            getattr(L, f).argtypes = [P, P]
        L.ovcs_destroy.argtypes = [P]
        L.ovcs_set_action.argtypes = [P, C.c_int32, C.c_int32]
        L.ovcs_step_instruction.argtypes = [P, C.c_int32]
        L.ovcs_tick.argtypes = [P, C.c_int32]
        L.ovcs_tick_trace.argtypes = [P, C.c_int32, C.c_int32, P, P]
        L.ovcs_get_debug.argtypes = [P, C.c_int32, C.POINTER(Debug)]
        L.ovcs_get_back.argtypes = [P, C.c_int32, P]
        L.ovcs_set_cpu.argtypes = [P] + [C.c_int32] * 7
        L.ovcs_poke_ram.argtypes = [P, C.c_int32, C.c_int32, C.c_int32]
        L.ovcs_alu_adc.argtypes = [C.c_int] * 3 + [C.POINTER(C.c_int)] * 2
        L.ovcs_alu_sbc.argtypes = [C.c_int] * 3 + [C.POINTER(C.c_int)] * 2
        L.ovcs_splitmix64.argtypes = [C.POINTER(C.c_uint64)]
        L.ovcs_splitmix64.restype = C.c_uint64
        L.ovcs_step_soft_range.argtypes = [P, P, C.c_int32, C.c_double, C.c_double, P, C.c_int32, C.c_int32]
        L.ovcs_soft_peek.argtypes = [P, C.c_int, C.c_int]; L.ovcs_soft_peek.restype = C.c_double
        L.ovcs_soft_peek_relaxed.argtypes = [P, C.c_int, C.c_int, C.c_double, C.c_int]; L.ovcs_soft_peek_relaxed.restype = C.c_double
        L.ovcs_soft_gate.argtypes = [C.c_double, C.c_int, C.c_double]; L.ovcs_soft_gate.restype = C.c_double
        L.ovcs_soft_ste.argtypes = [C.c_float, C.c_float]; L.ovcs_soft_ste.restype = C.c_float
        _lib = L
    return _lib


class OracleVCS:
    """Host-side batch of oracle consoles with the same surface as the CUDA binding."""

    def __init__(self, roms, seeds, env_rom=None, batch=None, y0=34, max_lines=320, f8_start_bank=1, mappers=None):
        L = lib()
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        self.batch = int(batch if batch is not None else len(seeds))
        self._rom_bufs = [(C.c_uint8 * len(r)).from_buffer_copy(bytes(r)) for r in roms]
        arr = (Rom * len(roms))()
        for i, b in enumerate(self._rom_bufs):
            arr[i].data = C.cast(b, C.POINTER(C.c_uint8)); arr[i].size = len(b)
            arr[i].mapper = 0 if mappers is None else (MAPPERS[mappers[i]] if isinstance(mappers[i], str) else int(mappers[i]))
        er = None if env_rom is None else np.ascontiguousarray(env_rom, dtype=np.int32)
        cfg = Config(y0, max_lines, f8_start_bank, 0)
        self.h = C.c_void_p()
        rc = L.ovcs_create(C.byref(self.h), self.batch, arr, len(roms),
                           None if er is None else er.ctypes.data, seeds.ctypes.data, C.byref(cfg))
        if rc != 0:
            raise RuntimeError(f"ovcs_create failed: {rc}")

    def close(self):
        if self.h:
            lib().ovcs_destroy(self.h); self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reset(self, mask=None):
        m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
        assert lib().ovcs_reset(self.h, None if m is None else m.ctypes.data) == 0

    def step(self, actions, frameskip=1, threads=1):
        a = np.ascontiguousarray(actions, dtype=np.uint8)
        assert a.shape == (self.batch,)
        if threads <= 1 or self.batch < 2:
            assert lib().ovcs_step(self.h, a.ctypes.data, frameskip) == 0
            return
        # envs are independent; ctypes releases the GIL, each thread runs the single-threaded oracle
        n = min(threads, self.batch)
        cuts = [self.batch * i // n for i in range(n + 1)]
        with ThreadPoolExecutor(n) as ex:
            rcs = list(ex.map(lambda i: lib().ovcs_step_range(self.h, a.ctypes.data, frameskip, cuts[i], cuts[i + 1]), range(n)))
        assert all(rc == 0 for rc in rcs)

    def step_instructions(self, actions, n_instr, threads=1):
        """latch the actions, then n_instr single-instruction steps per env (the paper's step unit)"""
        a = np.ascontiguousarray(actions, dtype=np.uint8)
        assert a.shape == (self.batch,)
        n = max(1, min(threads, self.batch))
        cuts = [self.batch * i // n for i in range(n + 1)]
        with ThreadPoolExecutor(n) as ex:
            rcs = list(ex.map(lambda i: lib().ovcs_step_instructions_range(self.h, a.ctypes.data, int(n_instr), cuts[i], cuts[i + 1]), range(n)))
        assert all(rc == 0 for rc in rcs)

    def step_instructions_soft(self, actions, n_instr, T, alpha, full, threads=1):
        """n_instr single-instruction steps per env in SOFT-STE (full False) or FULL mode (full True: the fully relaxed
        forward of PAPER.md appendix D).  Returns [batch][8] float64 as step_soft."""
        a = np.ascontiguousarray(actions, dtype=np.uint8)
        assert a.shape == (self.batch,)
        out = np.zeros((self.batch, 8), dtype=np.float64)
        n = max(1, min(threads, self.batch))
        cuts = [self.batch * i // n for i in range(n + 1)]
        with ThreadPoolExecutor(n) as ex:
            rcs = list(ex.map(lambda i: lib().ovcs_step_instructions_soft_range(self.h, a.ctypes.data, int(n_instr), float(T), float(alpha),
                                                                                 1 if full else 0, out.ctypes.data, cuts[i], cuts[i + 1]), range(n)))
        assert all(rc == 0 for rc in rcs)
        return out

    @staticmethod
    def _u8(x):
        return None if x is None else np.ascontiguousarray(x, dtype=np.uint8)

    def step_masked(self, actions, frameskip, mask, threads=1):
        a, m = self._u8(actions), self._u8(mask)
        mp = None if m is None else m.ctypes.data
        n = max(1, min(threads, self.batch))
        if n == 1:
            assert lib().ovcs_step_masked(self.h, a.ctypes.data, frameskip, mp) == 0
            return
        cuts = [self.batch * i // n for i in range(n + 1)]          # envs are independent: one oracle thread per slice
        with ThreadPoolExecutor(n) as ex:
            rcs = list(ex.map(lambda i: lib().ovcs_step_masked_range(self.h, a.ctypes.data, frameskip, mp, cuts[i], cuts[i + 1]), range(n)))
        assert all(rc == 0 for rc in rcs)

    def set_switches(self, switches=None):
        s = self._u8(switches)
        assert lib().ovcs_set_switches(self.h, None if s is None else s.ctypes.data) == 0

    def boot(self, mask=None, noop_frames=60, reset_frames=4, noop_starts=None, max_noop_starts=30, frameskip=4):
        m, k = self._u8(mask), self._u8(noop_starts)
        assert lib().ovcs_boot(self.h, None if m is None else m.ctypes.data, noop_frames, reset_frames,
                               None if k is None else k.ctypes.data, max_noop_starts, frameskip) == 0

    def step_soft(self, actions, frameskip, T, alpha, threads=1):
        """SOFT-STE forward step (config 5).  Returns [batch][8] float64: sum_rom, sum_ram, sum_gate, n_rom, n_ram,
        n_branch, mismatch, max_pull of this call."""
        a = np.ascontiguousarray(actions, dtype=np.uint8)
        assert a.shape == (self.batch,)
        out = np.zeros((self.batch, 8), dtype=np.float64)
        n = max(1, min(threads, self.batch))
        cuts = [self.batch * i // n for i in range(n + 1)]
        with ThreadPoolExecutor(n) as ex:
            rcs = list(ex.map(lambda i: lib().ovcs_step_soft_range(self.h, a.ctypes.data, frameskip, float(T), float(alpha),
                                                                    out.ctypes.data, cuts[i], cuts[i + 1]), range(n)))
        assert all(rc == 0 for rc in rcs)
        return out

    def ram(self):
        out = np.empty((self.batch, 128), dtype=np.uint8); assert lib().ovcs_get_ram(self.h, out.ctypes.data) == 0; return out

    def cart_ram(self):
        out = np.empty((self.batch, 128), dtype=np.uint8); assert lib().ovcs_get_cart_ram(self.h, out.ctypes.data) == 0; return out

    def regs(self):
        out = np.empty(self.batch, dtype=REGS_DTYPE); assert lib().ovcs_get_regs(self.h, out.ctypes.data) == 0; return out

    def screen(self):
        out = np.empty((self.batch, 210, 160), dtype=np.uint8); assert lib().ovcs_get_screen(self.h, out.ctypes.data) == 0; return out

    # ---- single-env test hooks
    def set_action(self, env, action): assert lib().ovcs_set_action(self.h, env, action) == 0
    def step_instruction(self, env=0): return lib().ovcs_step_instruction(self.h, env)
    def tick(self, env=0): assert lib().ovcs_tick(self.h, env) == 0
    def tick_trace(self, n, env=0):
        t = np.empty(n, dtype=np.uint8); f = np.empty(n, dtype=np.uint8)
        assert lib().ovcs_tick_trace(self.h, env, n, t.ctypes.data, f.ctypes.data) == 0
        return t, f
    def debug(self, env=0):
        d = Debug(); assert lib().ovcs_get_debug(self.h, env, C.byref(d)) == 0; return d
    def back(self, env=0):
        out = np.empty((210, 160), dtype=np.uint8); assert lib().ovcs_get_back(self.h, env, out.ctypes.data) == 0; return out
    def set_cpu(self, env=0, a=-1, x=-1, y=-1, sp=-1, p=-1, pc=-1): assert lib().ovcs_set_cpu(self.h, env, a, x, y, sp, p, pc) == 0
    def poke_ram(self, env, idx, value): assert lib().ovcs_poke_ram(self.h, env, idx, value) == 0


def detect_mapper(image: bytes) -> str:
    """ovcs_detect_mapper as a format name ('' when no format has that size)"""
    buf = (C.c_uint8 * len(image)).from_buffer_copy(bytes(image))
    k = lib().ovcs_detect_mapper(C.cast(buf, C.c_void_p), len(image))
    return {v: n for n, v in MAPPERS.items()}.get(k, "") if k > 0 else ""
