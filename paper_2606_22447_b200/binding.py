"""Thin ctypes binding over libvcsb200.so (include/vcs.h).  Argument marshalling only: every step of the
emulation runs in the CUDA kernels.  PyTorch supplies device memory and streams, nothing else.

There is no CPU fallback: if the shared library is missing, or no CUDA device is present, construction
raises.  This module never imports anything from oracle/.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_PKG, "libvcsb200.so")

VCS_OK, VCS_EINVAL, VCS_ECUDA, VCS_ENOMEM, VCS_EROM = 0, -1, -2, -3, -4
# vcs_config.flags (include/vcs.h): performance only, never results
VCS_F_NO_SPIN, VCS_F_NO_FUSE, VCS_F_NO_REGROUP, VCS_F_ROM_GLOBAL, VCS_F_NO_BALANCE, VCS_F_NO_PROMOTE = 1, 2, 4, 8, 16, 32
VCS_F_BLOCK_64, VCS_F_BLOCK_128, VCS_F_BLOCK_256 = 1 << 8, 2 << 8, 3 << 8
_ERR = {VCS_EINVAL: "VCS_EINVAL", VCS_ECUDA: "VCS_ECUDA", VCS_ENOMEM: "VCS_ENOMEM", VCS_EROM: "VCS_EROM"}

EXPORTS = ["vcs_create", "vcs_reset", "vcs_step", "vcs_step_instructions", "vcs_step_masked", "vcs_set_switches", "vcs_boot", "vcs_auto_reset", "vcs_get_booting", "vcs_step_soft", "vcs_step_instructions_soft", "vcs_get_ram", "vcs_get_regs", "vcs_get_cart_ram", "vcs_get_screen", "vcs_detect_mapper", "vcs_step_host", "vcs_step_host_noalloc",
           "vcs_get_ram_host", "vcs_get_regs_host", "vcs_get_screen_host", "vcs_screen_ptr", "vcs_block_times", "vcs_launch_count",
           "vcs_optable", "vcs_issue_peak", "vcs_destroy", "vcs_last_error"]

NOALLOC_MAX_BATCH = 65536        # VCS_NOALLOC_MAX_BATCH (include/vcs.h)

REGS_DTYPE = np.dtype([("cycles", "<u8"), ("frame", "<u4"), ("pc", "<u2"), ("a", "u1"), ("x", "u1"), ("y", "u1"),
                       ("sp", "u1"), ("p", "u1"), ("bank", "u1"), ("line", "<u2"), ("cyc_in_line", "u1"),
                       ("status", "u1"), ("intim", "u1"), ("timint", "u1"), ("pad", "u1", (6,))])
assert REGS_DTYPE.itemsize == 32


class VcsRom(C.Structure):
    _fields_ = [("data", C.POINTER(C.c_uint8)), ("size", C.c_uint32), ("mapper", C.c_uint32)]


MAPPERS = {"": 0, "2K": 1, "4K": 2, "F8": 3, "F6": 4, "F4": 5, "F8SC": 6, "F6SC": 7, "F4SC": 8, "E0": 9, "FE": 10}   # VCS_MAP_*


class VcsConfig(C.Structure):
    _fields_ = [("y0", C.c_int32), ("max_lines", C.c_int32), ("f8_start_bank", C.c_int32), ("flags", C.c_uint32)]


class VcsError(RuntimeError):
    pass


_lib = None


def load_library() -> C.CDLL:
    """dlopen libvcsb200.so; raises (never falls back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise VcsError(f"{_SO} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                       "(or paper_2606_22447_b200/build.py).  There is no CPU fallback.")
    L = C.CDLL(_SO)
    P = C.c_void_p
    L.vcs_create.argtypes = [C.POINTER(P), C.c_int32, C.POINTER(VcsRom), C.c_int32, P, P, C.POINTER(VcsConfig)]
    L.vcs_reset.argtypes = [P, P, P]
    L.vcs_step.argtypes = [P, P, C.c_int32, P]
    L.vcs_step_host.argtypes = [P, P, C.c_int32, P]
    L.vcs_step_host_noalloc.argtypes = [P, P, C.c_int32, P, P, P, P]
    L.vcs_step_instructions.argtypes = [P, P, C.c_int32, P]
    L.vcs_step_instructions_soft.argtypes = [P, P, C.c_int32, C.c_float, C.c_float, C.c_int32, P, P]
    L.vcs_step_masked.argtypes = [P, P, C.c_int32, P, P]
    L.vcs_set_switches.argtypes = [P, P, P]
    L.vcs_boot.argtypes = [P, P, C.c_int32, C.c_int32, P, C.c_int32, C.c_int32, P]
    L.vcs_auto_reset.argtypes = [P, P, C.c_int32, C.c_int32, P, C.c_int32, P]
    L.vcs_get_booting.argtypes = [P, P, P]
    L.vcs_step_soft.argtypes = [P, P, C.c_int32, C.c_float, C.c_float, P, P]
    L.vcs_detect_mapper.argtypes = [P, C.c_uint32]
    for f in ("vcs_get_ram", "vcs_get_regs", "vcs_get_cart_ram", "vcs_get_screen", "vcs_get_ram_host", "vcs_get_regs_host", "vcs_get_screen_host"):
        getattr(L, f).argtypes = [P, P, P]
    L.vcs_screen_ptr.argtypes = [P, C.POINTER(P)]
    L.vcs_block_times.argtypes = [P, P, P, C.c_int32, C.POINTER(C.c_int32)]
    L.vcs_launch_count.argtypes = [P]; L.vcs_launch_count.restype = C.c_int64
    L.vcs_optable.argtypes = [P]
    L.vcs_issue_peak.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.vcs_destroy.argtypes = [P]
    L.vcs_last_error.argtypes = [P]; L.vcs_last_error.restype = C.c_char_p
    _lib = L
    return L


def detect_mapper(image: bytes) -> str:
    """vcs_detect_mapper as a format name (host call; '' when no format has that size)"""
    buf = (C.c_uint8 * len(image)).from_buffer_copy(bytes(image))
    k = load_library().vcs_detect_mapper(C.cast(buf, C.c_void_p), len(image))
    return {v: n for n, v in MAPPERS.items()}.get(k, "") if k > 0 else ""


def optable() -> np.ndarray:
    out = np.zeros(256, dtype=np.uint16)
    assert load_library().vcs_optable(out.ctypes.data) == 0
    return out


def issue_peak(kind: int, iters: int = 4096) -> tuple[float, float]:
    """(thread-instructions/s, seconds) of the integer-issue micro-benchmark (vcs_issue_peak)."""
    v, sec = C.c_double(), C.c_double()
    rc = load_library().vcs_issue_peak(kind, iters, C.byref(v), C.byref(sec))
    if rc != 0:
        raise VcsError(f"vcs_issue_peak: {_ERR.get(rc, rc)}")
    return v.value, sec.value


def _stream_ptr(stream) -> int | None:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


class VCS:
    """A batch of consoles on the current CUDA device (vcs_create ... vcs_destroy)."""

    def __init__(self, roms, seeds, env_rom=None, y0=34, max_lines=320, f8_start_bank=1, flags=0, mappers=None):
        import torch
        if not torch.cuda.is_available():
            raise VcsError("no CUDA device: libvcsb200 has no CPU fallback")
        self.torch = torch
        L = self.L = load_library()
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        self.batch = int(seeds.shape[0])
        bufs = [(C.c_uint8 * len(r)).from_buffer_copy(bytes(r)) for r in roms]
        arr = (VcsRom * len(roms))()
        for i, b in enumerate(bufs):
            arr[i].data = C.cast(b, C.POINTER(C.c_uint8)); arr[i].size = len(b)
            arr[i].mapper = 0 if mappers is None else (MAPPERS[mappers[i]] if isinstance(mappers[i], str) else int(mappers[i]))
        er = None if env_rom is None else np.ascontiguousarray(env_rom, dtype=np.int32)
        cfg = VcsConfig(y0, max_lines, f8_start_bank, int(flags))
        self.h = C.c_void_p()
        rc = L.vcs_create(C.byref(self.h), self.batch, arr, len(roms), None if er is None else er.ctypes.data,
                          seeds.ctypes.data, C.byref(cfg))
        if rc != 0:
            msg = L.vcs_last_error(self.h).decode() if self.h else ""
            if self.h:
                L.vcs_destroy(self.h); self.h = C.c_void_p()
            raise VcsError(f"vcs_create: {_ERR.get(rc, rc)} {msg}")
        self.device = torch.device("cuda", torch.cuda.current_device())

    def _chk(self, rc, what):
        if rc != 0:
            raise VcsError(f"{what}: {_ERR.get(rc, rc)} {self.L.vcs_last_error(self.h).decode()}")

    def close(self):
        if getattr(self, "h", None):
            self.L.vcs_destroy(self.h); self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- device-pointer API (torch tensors carry the memory)
    def reset(self, mask=None, stream=None):
        ptr = None
        if mask is not None:
            assert mask.is_cuda and mask.dtype == self.torch.uint8 and mask.numel() == self.batch and mask.is_contiguous()
            ptr = mask.data_ptr()
        self._chk(self.L.vcs_reset(self.h, ptr, _stream_ptr(stream)), "vcs_reset")

    def step(self, actions, frameskip=4, stream=None):
        assert actions.is_cuda and actions.dtype == self.torch.uint8 and actions.numel() == self.batch and actions.is_contiguous()
        self._chk(self.L.vcs_step(self.h, actions.data_ptr(), int(frameskip), _stream_ptr(stream)), "vcs_step")

    def step_instructions(self, actions, n_instr, stream=None):
        """vcs_step_instructions: exactly n_instr CPU instructions per env (the paper's step unit); the screen is not updated."""
        assert actions.is_cuda and actions.dtype == self.torch.uint8 and actions.numel() == self.batch and actions.is_contiguous()
        self._chk(self.L.vcs_step_instructions(self.h, actions.data_ptr(), int(n_instr), _stream_ptr(stream)), "vcs_step_instructions")

    def step_instructions_soft(self, actions, n_instr, T, alpha, full, out=None, stream=None):
        """vcs_step_instructions_soft: n_instr instructions per env in SOFT-STE (full False) or FULL mode (full True, the
        fully relaxed forward); returns the device float[batch][8] of per-env soft sums."""
        t = self.torch
        assert actions.is_cuda and actions.dtype == t.uint8 and actions.numel() == self.batch and actions.is_contiguous()
        out = t.empty((self.batch, 8), dtype=t.float32, device=self.device) if out is None else out
        self._chk(self.L.vcs_step_instructions_soft(self.h, actions.data_ptr(), int(n_instr), float(T), float(alpha), 1 if full else 0,
                                                    out.data_ptr(), _stream_ptr(stream)), "vcs_step_instructions_soft")
        return out

    def _u8(self, x, what):
        if x is None:
            return None
        assert x.is_cuda and x.dtype == self.torch.uint8 and x.numel() == self.batch and x.is_contiguous(), what
        return x.data_ptr()

    def step_masked(self, actions, frameskip, mask, stream=None):
        """vcs_step_masked: envs with mask == 0 stay frozen."""
        self._chk(self.L.vcs_step_masked(self.h, self._u8(actions, "actions"), int(frameskip), self._u8(mask, "mask"),
                                         _stream_ptr(stream)), "vcs_step_masked")

    def set_switches(self, switches=None, stream=None):
        """vcs_set_switches: SWCHB input pins per env (None = the default 0x3F)."""
        self._chk(self.L.vcs_set_switches(self.h, self._u8(switches, "switches"), _stream_ptr(stream)), "vcs_set_switches")

    def boot(self, mask=None, noop_frames=60, reset_frames=4, noop_starts=None, max_noop_starts=30, frameskip=4, stream=None):
        """vcs_boot: ALE-style episode start (reset, NOOP frames, RESET-switch frames, per-env NOOP steps)."""
        self._chk(self.L.vcs_boot(self.h, self._u8(mask, "mask"), int(noop_frames), int(reset_frames),
                                  self._u8(noop_starts, "noop_starts"), int(max_noop_starts), int(frameskip),
                                  _stream_ptr(stream)), "vcs_boot")

    def auto_reset(self, mask=None, noop_steps=15, reset_steps=1, noop_starts=None, max_noop_starts=30, stream=None):
        """vcs_auto_reset: reset + arm the masked envs; their boot runs inside the following step calls."""
        self._chk(self.L.vcs_auto_reset(self.h, self._u8(mask, "mask"), int(noop_steps), int(reset_steps),
                                        self._u8(noop_starts, "noop_starts"), int(max_noop_starts), _stream_ptr(stream)),
                  "vcs_auto_reset")

    def get_booting(self, out=None, stream=None):
        t = self.torch
        out = t.empty(self.batch, dtype=t.uint8, device=self.device) if out is None else out
        self._chk(self.L.vcs_get_booting(self.h, out.data_ptr(), _stream_ptr(stream)), "vcs_get_booting"); return out

    def step_soft(self, actions, frameskip, T, alpha, out=None, stream=None):
        """SOFT-STE forward step (vcs_step_soft); returns the device float[batch][8] of per-env soft sums."""
        t = self.torch
        assert actions.is_cuda and actions.dtype == t.uint8 and actions.numel() == self.batch and actions.is_contiguous()
        out = t.empty((self.batch, 8), dtype=t.float32, device=self.device) if out is None else out
        self._chk(self.L.vcs_step_soft(self.h, actions.data_ptr(), int(frameskip), float(T), float(alpha), out.data_ptr(),
                                       _stream_ptr(stream)), "vcs_step_soft")
        return out

    def get_ram(self, out=None, stream=None):
        t = self.torch
        out = t.empty((self.batch, 128), dtype=t.uint8, device=self.device) if out is None else out
        self._chk(self.L.vcs_get_ram(self.h, out.data_ptr(), _stream_ptr(stream)), "vcs_get_ram"); return out

    def get_cart_ram(self, out=None, stream=None):
        t = self.torch
        out = t.empty((self.batch, 128), dtype=t.uint8, device=self.device) if out is None else out
        self._chk(self.L.vcs_get_cart_ram(self.h, out.data_ptr(), _stream_ptr(stream)), "vcs_get_cart_ram"); return out

    def get_regs(self, out=None, stream=None):
        t = self.torch
        out = t.empty((self.batch, 32), dtype=t.uint8, device=self.device) if out is None else out
        self._chk(self.L.vcs_get_regs(self.h, out.data_ptr(), _stream_ptr(stream)), "vcs_get_regs"); return out

    def get_screen(self, out=None, stream=None):
        t = self.torch
        out = t.empty((self.batch, 210, 160), dtype=t.uint8, device=self.device) if out is None else out
        self._chk(self.L.vcs_get_screen(self.h, out.data_ptr(), _stream_ptr(stream)), "vcs_get_screen"); return out

    # ---- host-pointer API (numpy in / out; the copies happen inside the C call)
    def step_host(self, actions: np.ndarray, frameskip=4, stream=None):
        a = np.ascontiguousarray(actions, dtype=np.uint8); assert a.shape == (self.batch,)
        self._chk(self.L.vcs_step_host(self.h, a.ctypes.data, int(frameskip), _stream_ptr(stream)), "vcs_step_host")

    def step_host_noalloc(self, actions: np.ndarray, frameskip=4, ram_out=None, regs_out=None, flagged_out=None, stream=None, sync=True):
        """vcs_step_host_noalloc: step + read-back of RAM / regs / number of envs with a status bit, staged in the library's
        static device array (no allocation on the CUDA side; batch <= NOALLOC_MAX_BATCH).  The C call only enqueues: with
        sync=True the stream is synchronised here and (ram, regs, n_flagged) are returned ready to read."""
        a = np.ascontiguousarray(actions, dtype=np.uint8); assert a.shape == (self.batch,)
        ram = np.empty((self.batch, 128), dtype=np.uint8) if ram_out is None else ram_out
        regs = np.empty(self.batch, dtype=REGS_DTYPE) if regs_out is None else regs_out
        flagged = np.full(1, -1, dtype=np.int32) if flagged_out is None else flagged_out
        sp = _stream_ptr(stream)
        self._keep = (a, ram, regs, flagged)                # the buffers must outlive the enqueued copies
        self._chk(self.L.vcs_step_host_noalloc(self.h, a.ctypes.data, int(frameskip), ram.ctypes.data, regs.ctypes.data, flagged.ctypes.data, sp),
                  "vcs_step_host_noalloc")
        if sync:
            (self.torch.cuda.current_stream() if stream is None else stream).synchronize()
        return ram, regs, flagged

    def ram_host(self, stream=None) -> np.ndarray:
        out = np.empty((self.batch, 128), dtype=np.uint8)
        self._chk(self.L.vcs_get_ram_host(self.h, out.ctypes.data, _stream_ptr(stream)), "vcs_get_ram_host"); return out

    def regs_host(self, stream=None) -> np.ndarray:
        out = np.empty(self.batch, dtype=REGS_DTYPE)
        self._chk(self.L.vcs_get_regs_host(self.h, out.ctypes.data, _stream_ptr(stream)), "vcs_get_regs_host"); return out

    def screen_host(self, out=None, stream=None) -> np.ndarray:
        out = np.empty((self.batch, 210, 160), dtype=np.uint8) if out is None else out
        self._chk(self.L.vcs_get_screen_host(self.h, out.ctypes.data, _stream_ptr(stream)), "vcs_get_screen_host"); return out

    def block_times(self):
        """(times uint64[n][3] = start ns, end ns, SM id of each block of the last plain step; perm int32[n])."""
        n = C.c_int32(0)
        self._chk(self.L.vcs_block_times(self.h, None, None, 0, C.byref(n)), "vcs_block_times")
        times = np.zeros((n.value, 3), dtype=np.uint64); perm = np.zeros(n.value, dtype=np.int32)
        self._chk(self.L.vcs_block_times(self.h, times.ctypes.data, perm.ctypes.data, n.value, C.byref(n)), "vcs_block_times")
        return times, perm

    def launch_count(self) -> int:
        return int(self.L.vcs_launch_count(self.h))
