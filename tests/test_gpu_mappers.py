"""CUDA path vs oracle on F6 / F4 cartridges: bit-exact RAM, regs, screens."""
import os

import numpy as np
import pytest

from test_gpu_parity import compare, torch  # noqa: F401
from test_oracle_mappers import banked_image
from vcs_inputs import SplitMix64, env_seeds
from vcs_inputs.romgen import FEATURES, make_rom

pytestmark = pytest.mark.gpu
NCPU = os.cpu_count() or 1


def pair(roms, seeds, env_rom=None, **kw):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    return VCS(roms, seeds, env_rom, **kw), OracleVCS(roms, seeds, env_rom, **kw)


def run(torch, roms, env_rom, steps, tag, frameskip=4):
    n = len(env_rom)
    g, o = pair(roms, env_seeds(31, n), np.asarray(env_rom, np.int32))
    r = SplitMix64(1234 + n)
    compare(g, o, f"{tag} reset")
    for t in range(steps):
        a = np.array([r.rnd(18) for _ in range(n)], np.uint8)
        g.step(torch.from_numpy(a).cuda(), frameskip); o.step(a, frameskip, threads=NCPU)
        compare(g, o, f"{tag} step {t}")
    banks = g.regs_host()["bank"]
    g.close(); o.close()
    return banks


@pytest.mark.parametrize("kind,nb", [("f6", 4), ("f4", 8)])
def test_generated_roms_one_mapper(torch, kind, nb):
    roms = [make_rom(900 + k, FEATURES[kind]) for k in range(2)]
    banks = run(torch, roms, [e // 80 for e in range(160)], 10, kind)     # blocks that share a ROM, ragged last block
    assert banks.max() < nb and len(set(banks.tolist())) > 2              # the random bank jumps really spread the envs


def test_mixed_mappers_in_one_batch(torch):
    roms = [make_rom(7, FEATURES["4a"]), make_rom(8, FEATURES["4b"]), make_rom(9, FEATURES["f6"]), make_rom(10, FEATURES["f4"]),
            make_rom(11, FEATURES[1])]
    run(torch, roms, [(e * 7) % 5 for e in range(150)], 8, "mixed")      # every lane of a warp on another cartridge


@pytest.mark.parametrize("nb,lo", [(4, 0xFFF6), (8, 0xFFF4)])
def test_hotspot_program(torch, nb, lo):
    def build(a):
        a.org(0xF000); a.op("LDX", "imm", 0xFF); a.op("TXS")
        for k in range(nb):
            a.op("LDA", "abs", lo + k); a.op("STA", "zp", 0x80 + k); a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x90 + k)
        a.op("STA", "abs", lo + nb - 1); a.op("LDA", "abs", lo - 1); a.op("LDA", "abs", lo + nb)
        a.op("LDX", "imm", 0xFF); a.op("LDA", "abx", lo + 1 - 0xFF); a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0xA0)
        a.op("LDY", "imm", 0x10); a.op("STA", "aby", lo - 0x10); a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0xA1)
        a.op("LDA", "imm", 2); a.op("STA", "zp", 0x00); a.op("LDA", "imm", 0); a.op("STA", "zp", 0x00)     # VSYNC on/off: a frame end
        a.op("JMP", "abs", 0xF003)
    img = banked_image(build, nb)
    g, o = pair([img], env_seeds(5, 40))
    for t in range(4):
        a = np.zeros(40, np.uint8)
        g.step(torch.from_numpy(a).cuda(), 1 + t); o.step(a, 1 + t)
        compare(g, o, f"hotspots nb={nb} step {t}")
    assert g.ram_host()[0, 0x10:0x10 + nb].tolist() == [0xA0 + k for k in range(nb)]


def test_soft_mode_on_f6(torch):
    roms = [make_rom(77, FEATURES["f6"])]
    n = 48
    g, o = pair(roms, env_seeds(9, n))
    r = SplitMix64(4)
    for t in range(3):
        a = np.array([r.rnd(18) for _ in range(n)], np.uint8)
        g.step_soft(torch.from_numpy(a).cuda(), 2, 1.0, 4.0); o.step(a, 2, threads=NCPU)     # Theorem 1/3: soft forward == hard
        compare(g, o, f"soft f6 step {t}")
