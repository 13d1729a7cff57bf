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
    okw = {k: v for k, v in kw.items() if k != "flags"}
    return VCS(roms, seeds, env_rom, **kw), OracleVCS(roms, seeds, env_rom, **okw)


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


# ---------------------------------------------------------------------------------------------- Superchip, E0, FE
from vcs_inputs import superchip_rom, e0_rom, fe_rom


def compare_cart_ram(g, o, tag):
    assert (g.get_cart_ram().cpu().numpy() == o.cart_ram()).all(), f"{tag}: Superchip RAM differs"


def run_kinds(torch, roms, kinds, env_rom, steps, tag, **kw):
    n = len(env_rom)
    g, o = pair(roms, env_seeds(37, n), np.asarray(env_rom, np.int32), mappers=kinds, **kw)
    r = SplitMix64(99 + n)
    compare(g, o, f"{tag} reset"); compare_cart_ram(g, o, f"{tag} reset")
    for t in range(steps):
        a = np.array([r.rnd(18) for _ in range(n)], np.uint8)
        fs = 1 + t % 3
        g.step(torch.from_numpy(a).cuda(), fs); o.step(a, fs, threads=NCPU)
        compare(g, o, f"{tag} step {t}"); compare_cart_ram(g, o, f"{tag} step {t}")
    regs = g.regs_host()
    g.close(); o.close()
    return regs


@pytest.mark.parametrize("kind", ["F8SC", "F6SC", "F4SC"])
def test_superchip_carts(torch, kind):
    regs = run_kinds(torch, [superchip_rom(kind, 21), superchip_rom(kind, 22)], [kind, kind], [e // 72 for e in range(144)], 8, kind, max_lines=200)
    assert (regs["status"] == 0).all() and len(set(regs["bank"].tolist())) > 1


def test_e0_carts(torch):
    regs = run_kinds(torch, [e0_rom(31), e0_rom(32)], ["E0", "E0"], [e // 72 for e in range(144)], 8, "E0", max_lines=200)
    assert (regs["status"] == 0).all() and len(set(zip(regs["bank"].tolist(), regs["pad"][:, 0].tolist()))) > 4


def test_fe_carts(torch):
    regs = run_kinds(torch, [fe_rom(41), fe_rom(42)], ["FE", "FE"], [e // 72 for e in range(144)], 8, "FE", max_lines=200)
    assert (regs["status"] == 0).all()


def test_all_ten_formats_in_one_batch(torch):
    """every lane of a warp on a cartridge of another format, the Superchip program also run as a plain F8 image (no RAM there)"""
    roms = [make_rom(7, FEATURES[1]), make_rom(8, FEATURES["4a"]), make_rom(9, FEATURES["4b"]), make_rom(10, FEATURES["f6"]), make_rom(11, FEATURES["f4"]),
            superchip_rom("F8SC", 51), superchip_rom("F6SC", 52), superchip_rom("F4SC", 53), e0_rom(54), fe_rom(55), superchip_rom("F8SC", 51)]
    kinds = ["2K", "4K", "F8", "F6", "F4", "F8SC", "F6SC", "F4SC", "E0", "FE", "F8"]
    run_kinds(torch, roms, kinds, [(e * 5) % 11 for e in range(165)], 8, "ten formats", max_lines=220)


def test_special_formats_instruction_steps_and_blocks(torch):
    """the same carts in 256-env blocks that share a ROM (staged in shared memory), and stepped by instructions"""
    from paper_2606_22447_b200.binding import VCS_F_BLOCK_256
    roms = [superchip_rom("F8SC", 61), e0_rom(62), fe_rom(63)]; kinds = ["F8SC", "E0", "FE"]
    env_rom = [e // 256 for e in range(768)]
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    seeds = env_seeds(5, 768)
    g = VCS(roms, seeds, np.asarray(env_rom, np.int32), mappers=kinds, max_lines=200, flags=VCS_F_BLOCK_256)
    o = OracleVCS(roms, seeds, np.asarray(env_rom, np.int32), mappers=kinds, max_lines=200)
    r = SplitMix64(3)
    for t in range(4):
        a = np.array([r.rnd(18) for _ in range(768)], np.uint8)
        g.step(torch.from_numpy(a).cuda(), 2); o.step(a, 2, threads=NCPU)
        compare(g, o, f"special blocks step {t}"); compare_cart_ram(g, o, f"special blocks step {t}")
    for n in (1, 13, 700):
        a = np.array([r.rnd(18) for _ in range(768)], np.uint8)
        g.step_instructions(torch.from_numpy(a).cuda(), n); o.step_instructions(a, n, threads=NCPU)
        gr, orr = g.regs_host(), o.regs()
        for f in gr.dtype.names:
            assert (gr[f] == orr[f]).all(), f"instructions {n}: regs.{f}"
        assert (g.ram_host() == o.ram()).all(); compare_cart_ram(g, o, f"instructions {n}")


def test_format_errors(torch):
    from paper_2606_22447_b200 import VCS, VcsError
    with pytest.raises(VcsError):
        VCS([bytes(4096)], env_seeds(1, 4), mappers=["E0"])                         # E0 is an 8 KB format
    with pytest.raises(VcsError):
        VCS([bytes(8192)], env_seeds(1, 4), mappers=[77])
    g = VCS([e0_rom(1)], env_seeds(1, 4), mappers=["E0"])
    with pytest.raises(VcsError):
        g.step_soft(torch.zeros(4, dtype=torch.uint8, device="cuda"), 1, 1.0, 4.0)   # hard mode only


# ---- blocks that hold ONE banked cartridge regroup their envs at bank switches: F6 / F4 with
# four / eight banks (the image read from global memory, classes padded to warp boundaries while the spare warp's lanes
# last) and the Superchip variants.  Which thread runs which env never shows in the results.
@pytest.mark.parametrize("kind,nb", [("f6", 4), ("f4", 8)])
@pytest.mark.parametrize("flags", ["VCS_F_BLOCK_64", "VCS_F_BLOCK_128", "VCS_F_BLOCK_256", "VCS_F_BLOCK_128|VCS_F_NO_REGROUP"])
def test_one_banked_rom_per_block_regroups(torch, kind, nb, flags):
    import paper_2606_22447_b200.binding as b
    fl = 0
    for f in flags.split("|"): fl |= getattr(b, f)
    n = 300                                                               # full blocks and a ragged last one at every block size
    g, o = pair([make_rom(940 + nb, FEATURES[kind])], env_seeds(41, n), flags=fl)
    r = SplitMix64(77 + nb)
    for t in range(8):
        a = np.array([r.rnd(18) for _ in range(n)], np.uint8)
        g.step(torch.from_numpy(a).cuda(), 3); o.step(a, 3, threads=NCPU)
        compare(g, o, f"{kind} {flags} step {t}")
    banks = g.regs_host()["bank"]
    assert banks.max() < nb and len(set(banks.tolist())) > 2
    g.close(); o.close()


@pytest.mark.parametrize("kind", ["F8SC", "F6SC", "F4SC"])
def test_one_superchip_rom_per_block_regroups(torch, kind):
    import paper_2606_22447_b200.binding as b
    regs = run_kinds(torch, [superchip_rom(kind, 23)], [kind], [0] * 300, 9, kind + " one rom", max_lines=200, flags=b.VCS_F_BLOCK_128)
    assert len(set(regs["bank"].tolist())) > 1
