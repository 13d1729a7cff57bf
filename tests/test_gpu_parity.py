"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, bit-exact.

RAM (128 B), every vcs_regs field (registers, cycle counter, beam, bank, status, timer) and the 160x210
palette-index screen are compared after every step (PAPER.md L167 exactness metrics; L592 batched ==
unbatched).  Inputs are the seeded synthetic configs of SURVEY §8(d) G.2 at sizes the oracle finishes in
seconds, plus BASELINE's full batch with a sampled subset of envs."""
import os

import numpy as np
import pytest

from vcs_inputs import make_workload, hand_rom, SplitMix64, TIA_W, RIOT, env_seeds

pytestmark = pytest.mark.gpu
NCPU = os.cpu_count() or 1


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def mk(torch, w, **kw):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    return VCS(w.roms, w.seeds, w.env_rom, **kw), OracleVCS(w.roms, w.seeds, w.env_rom, **kw)


def compare(g, o, tag, envs=None, osel=None):
    """g: CUDA batch; o: oracle batch.  envs: indices into g to compare against all of o (sampling)."""
    gram, gregs, gscr = g.ram_host(), g.regs_host(), g.screen_host()
    if envs is not None:
        gram, gregs, gscr = gram[envs], gregs[envs], gscr[envs]
    oram, oregs, oscr = o.ram(), o.regs(), o.screen()
    for f in gregs.dtype.names:
        bad = np.nonzero((gregs[f] != oregs[f]).reshape(len(oregs), -1).any(axis=1))[0]
        assert bad.size == 0, f"{tag}: regs.{f} differs for envs {bad[:8]}: gpu {gregs[f][bad[:4]]} oracle {oregs[f][bad[:4]]}"
    bad = np.nonzero((gram != oram).any(axis=1))[0]
    assert bad.size == 0, f"{tag}: RAM differs for envs {bad[:8]}"
    bad = np.nonzero((gscr != oscr).any(axis=(1, 2)))[0]
    if bad.size:
        e = bad[0]; ys, xs = np.nonzero(gscr[e] != oscr[e])
        raise AssertionError(f"{tag}: screen differs for envs {bad[:8]}; env {e}: {ys.size} px, first (row {ys[0]}, x {xs[0]}) "
                             f"gpu {gscr[e][ys[0], xs[0]]} oracle {oscr[e][ys[0], xs[0]]}")


def run_parity(torch, w, steps, frameskip=None, tag="", **kw):
    g, o = mk(torch, w, **kw)
    fs = w.frameskip if frameskip is None else frameskip
    acts = w.actions(0, steps)
    compare(g, o, f"{tag} reset")
    for t in range(steps):
        g.step(torch.from_numpy(acts[t]).cuda(), fs)
        o.step(acts[t], fs, threads=NCPU)
        compare(g, o, f"{tag} step {t}")
    g.close(); o.close()


def test_config1_full(torch):
    """config 1 exactly as BASELINE.json states it: 1 env, 2 KB ROM, 10 frames, NOOP, compare per frame."""
    run_parity(torch, make_workload(1), 10, tag="config1")


def test_config2_every_env_every_step(torch):
    run_parity(torch, make_workload(2, batch=160), 12, tag="config2")      # 160 = one full block + a ragged tail


def test_config3_features(torch):
    run_parity(torch, make_workload(3, batch=96), 10, tag="config3")


def test_config4_heterogeneous_roms_and_f8(torch):
    run_parity(torch, make_workload(4, batch=256, n_roms=32), 8, tag="config4")


@pytest.mark.parametrize("fs", [1, 2, 3, 5])
def test_frameskips(torch, fs):
    run_parity(torch, make_workload(3, batch=40), 6, frameskip=fs, tag=f"frameskip{fs}")


def test_other_y0_and_cap(torch):
    run_parity(torch, make_workload(2, batch=33), 4, tag="y0=2", y0=2)
    run_parity(torch, make_workload(2, batch=33), 4, tag="y0=60,cap=200", y0=60, max_lines=200)   # cap ends frames mid-picture
    run_parity(torch, make_workload(4, batch=32, n_roms=4), 4, tag="bank0", f8_start_bank=0)


def test_batched_equals_unbatched(torch):
    """env e inside a batch == env e alone."""
    from paper_2606_22447_b200 import VCS
    w = make_workload(3, batch=200)
    acts = w.actions(0, 5)
    g = VCS(w.roms, w.seeds, w.env_rom)
    for t in range(5):
        g.step(torch.from_numpy(acts[t]).cuda(), 4)
    ram, regs, scr = g.ram_host(), g.regs_host(), g.screen_host()
    for e in (0, 77, 199):
        g1 = VCS(w.roms, w.seeds[e:e + 1], w.env_rom[e:e + 1])
        for t in range(5):
            g1.step(torch.from_numpy(acts[t][e:e + 1].copy()).cuda(), 4)
        assert (g1.ram_host()[0] == ram[e]).all() and g1.regs_host()[0] == regs[e] and (g1.screen_host()[0] == scr[e]).all()


def test_reset_mask_and_device_getters(torch):
    w = make_workload(2, batch=64)
    g, o = mk(torch, w)
    acts = w.actions(0, 4)
    for t in range(2):
        g.step(torch.from_numpy(acts[t]).cuda(), 4); o.step(acts[t], 4, threads=NCPU)
    mask = (np.arange(64) % 3 == 0).astype(np.uint8)
    g.reset(torch.from_numpy(mask).cuda()); o.reset(mask)
    compare(g, o, "after masked reset")
    for t in range(2, 4):
        g.step(torch.from_numpy(acts[t]).cuda(), 4); o.step(acts[t], 4, threads=NCPU)
        compare(g, o, f"masked reset step {t}")
    # device-pointer getters agree with the host-pointer ones
    assert (g.get_ram().cpu().numpy() == g.ram_host()).all()
    assert (g.get_screen().cpu().numpy() == g.screen_host()).all()
    assert (g.get_regs().cpu().numpy().view(g.regs_host().dtype).reshape(-1) == g.regs_host()).all()
    # host-pointer step == device-pointer step
    g2, _ = mk(torch, w)
    for t in range(2):
        g2.step_host(acts[t], 4)
    g3, _ = mk(torch, w)
    for t in range(2):
        g3.step(torch.from_numpy(acts[t]).cuda(), 4)
    assert (g2.ram_host() == g3.ram_host()).all() and (g2.screen_host() == g3.screen_host()).all()


def _chaos_rom(seed: int) -> bytes:
    """Unstructured TIA/RIOT torture: stores and RMWs to every TIA register at arbitrary beam positions,
    lines crossed mid-instruction, WSYNC/HMOVE/RESxx/VSYNC/VBLANK at random, collision and timer reads.
    Frames end by VSYNC toggles or by the cap.  Exercises the lazy TIA against the per-clock oracle."""
    r = SplitMix64(seed)
    regs = [n for n in TIA_W if not n.startswith("AUD")]

    def build(a):
        a.org(0xF000); a.op("LDX", "imm", 0xFF); a.op("TXS")
        a.label("top")
        for _ in range(330):
            k = r.rnd(20)
            if k < 9:
                reg = r.choice(regs)
                if reg in ("VSYNC", "WSYNC") and r.chance(2, 3): reg = r.choice(["GRP0", "GRP1", "PF1", "COLUBK", "ENABL", "ENAM0"])
                a.op(r.choice(["LDA", "LDX", "LDY"]), "imm", r.rnd(256)) if r.chance(2, 3) else None
                a.op(r.choice(["STA", "STX", "STY"]), "zp", TIA_W[reg])
            elif k < 11:
                a.op(r.choice(["INC", "DEC", "ASL", "LSR", "ROL", "ROR"]), "zp", TIA_W[r.choice(regs)])    # RMW on the TIA: two writes
            elif k < 13:
                a.op(r.choice(["LDA", "ADC", "EOR", "ORA"]), "zp", r.rnd(16)); a.op("STA", "zp", 0x80 + r.rnd(64))   # CXxx / INPTx reads
            elif k < 14:
                a.op("LDA", "imm", r.rnd(256)); a.op("STA", "abs", RIOT[r.choice(["TIM1T", "TIM8T", "TIM64T", "T1024T"])])
            elif k < 16:
                a.op("LDA", "abs", RIOT[r.choice(["INTIM", "TIMINT", "SWCHA", "SWCHB"])]); a.op("STA", "zp", 0x80 + r.rnd(64))
            elif k < 17:
                a.op("LDA", "imm", r.rnd(256)); a.op("STA", "abs", RIOT[r.choice(["SWACNT", "SWCHA", "SWBCNT", "SWCHB"])])
            elif k < 18:
                a.op("LDA", "abx", RIOT["INTIM"] - 0x20 + r.rnd(0x40)); a.op("INX")       # indexed: dummy/real reads around the RIOT
            else:
                if r.chance(1, 3): a.op("PHA"); a.op("PLA")
                elif r.chance(1, 4):                              # the stack on TIA registers: pushes are register writes, pulls read latches
                    a.op("LDX", "imm", r.rnd(0x80)); a.op("TXS"); a.op(r.choice(["PHA", "PHP"])); a.op(r.choice(["PHA", "PLA", "PLP"])); a.op("LDX", "imm", 0xFF); a.op("TXS")
                else: a.op(r.choice(["NOP", "INX", "DEY", "CLC", "SEC"]))
        a.op("JMP", "abs", "top")
    return hand_rom(build)


@pytest.mark.parametrize("seed", range(6))
def test_chaos_tia_riot(torch, seed):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    rom = _chaos_rom(1000 + seed)
    seeds = env_seeds(50 + seed, 48)
    kw = dict(max_lines=120 + 37 * seed, y0=2 + 5 * seed)
    g, o = VCS([rom], seeds, **kw), OracleVCS([rom], seeds, **kw)
    rng = SplitMix64(seed)
    for t in range(10):
        a = np.array([rng.rnd(20) for _ in range(48)], np.uint8)          # includes out-of-range actions (-> NOOP)
        fs = 1 + t % 3
        g.step(torch.from_numpy(a).cuda(), fs); o.step(a, fs, threads=NCPU)
        compare(g, o, f"chaos{seed} step {t}")


def test_illegal_opcode_and_cap(torch):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS

    def build(a):
        a.org(0xF000); a.op("LDA", "imm", 0x4C); a.op("STA", "zp", TIA_W["COLUBK"]); a.op("INC", "zp", 0x80)
        a.op("LDA", "zp", 0x80); a.op("CMP", "imm", 7); a.op("BNE", "rel", -12); a.byte(0x02)     # KIL after a few loops
    rom = hand_rom(build)
    seeds = env_seeds(9, 5)
    g, o = VCS([rom], seeds, max_lines=64), OracleVCS([rom], seeds, max_lines=64)
    for t in range(4):
        a = np.zeros(5, np.uint8)
        g.step(torch.from_numpy(a).cuda(), 2); o.step(a, 2)
        compare(g, o, f"illegal step {t}")
    assert (g.regs_host()["status"] & 1).all()


def test_full_batch_sampled(torch):
    """BASELINE config 4 at its full size and in bench.py's launch configuration (65,536 envs, 256 ROMs,
    frameskip 4): one env per ROM is checked against the oracle after every step."""
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    w = make_workload(4)
    g = VCS(w.roms, w.seeds, w.env_rom)
    idx = np.arange(256) * 256 + (np.arange(256) * 37) % 256           # one env per ROM, varying lane/warp
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    acts = w.actions(0, 3)
    for t in range(3):
        g.step(torch.from_numpy(acts[t]).cuda(), 4)
        o.step(acts[t][idx], 4, threads=NCPU)
        compare(g, o, f"config4 full step {t}", envs=idx)
    r = g.regs_host()
    assert (r["status"] == 0).all() and (r["frame"] == 12).all()
    assert (abs(r["cycles"].astype(np.int64) - 11 * 19912) < 19912).all()  # every frame is a 262-line NTSC frame (first one starts at reset)


def _spin_rom(seed: int) -> bytes:
    """Timer wait loops in every regime the closed-form fast-forward (HC_SPIN) must get right or hand back to the
    plain interpreter: all four divisors, INTIM polls that can step over the single cycle TIM1T shows 0, polls started
    after the underflow, waits with the picture on (line ends render), waits that run into the frame cap."""
    r = SplitMix64(seed)

    def build(a):
        a.org(0xF000); a.op("LDX", "imm", 0xFF); a.op("TXS")
        a.label("top")
        for i in range(40):
            div = r.choice(["TIM1T", "TIM8T", "TIM64T", "T1024T"])
            val = r.rnd(256) if div != "T1024T" else r.rnd(6)
            if r.chance(1, 2):                                    # picture on or off during the wait
                a.op("LDA", "imm", r.choice([0, 2])); a.op("STA", "zp", TIA_W["VBLANK"])
                a.op("LDA", "imm", r.rnd(256)); a.op("STA", "zp", TIA_W[r.choice(["PF1", "GRP0", "COLUBK", "ENABL"])])
            for _ in range(r.rnd(4)): a.op("NOP")
            a.op("LDA", "imm", val); a.op("STA", "abs", RIOT[div])
            if r.chance(1, 4):                                    # let it underflow first: the flag is already set when the poll starts
                a.op("LDY", "imm", 40 + r.rnd(200)); d = a.newlabel("D"); a.label(d); a.op("DEY"); a.op("BNE", "rel", d)
            for _ in range(r.rnd(5)): a.op("NOP")
            w = a.newlabel("W"); a.label(w)
            if r.chance(1, 2): a.op("LDA", "abs", RIOT["INTIM"]); a.op("BNE", "rel", w)
            else: a.op("BIT", "abs", RIOT["TIMINT"]); a.op("BPL", "rel", w)
            a.op("STA", "zp", 0x80 + i); a.op("PHP"); a.op("PLA"); a.op("STA", "zp", 0xC0 + (i & 31))
            if r.chance(1, 5): a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VSYNC"]); a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VSYNC"])
        a.op("JMP", "abs", "top")
    return hand_rom(build)


@pytest.mark.parametrize("seed", range(4))
def test_timer_wait_loops(torch, seed):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    rom = _spin_rom(2000 + seed)
    seeds = env_seeds(70 + seed, 40)
    kw = dict(max_lines=90 + 60 * seed)                          # small caps: waits run into the frame cap
    g, o = VCS([rom], seeds, **kw), OracleVCS([rom], seeds, **kw)
    for t in range(8):
        a = np.zeros(40, np.uint8)
        fs = 1 + t % 4
        g.step(torch.from_numpy(a).cuda(), fs); o.step(a, fs, threads=NCPU)
        compare(g, o, f"spin{seed} step {t}")


class _DevCompare:
    """compare a subset of a big CUDA batch with an oracle batch without moving the whole batch to the host: the
    getters fill device buffers once allocated here, the subset is gathered on the device"""
    def __init__(self, torch, g, idx):
        self.t, self.g = torch, g
        self.idx = torch.from_numpy(np.asarray(idx, dtype=np.int64)).cuda()
        self.ram = torch.empty((g.batch, 128), dtype=torch.uint8, device="cuda")
        self.regs = torch.empty((g.batch, 32), dtype=torch.uint8, device="cuda")
        self.scr = torch.empty((g.batch, 210, 160), dtype=torch.uint8, device="cuda")

    def check(self, o, tag, screens=True):
        from paper_2606_22447_b200.binding import REGS_DTYPE
        g = self.g
        gram = g.get_ram(self.ram)[self.idx].cpu().numpy()
        gregs = g.get_regs(self.regs)[self.idx].cpu().numpy().view(REGS_DTYPE).reshape(-1)
        oram, oregs = o.ram(), o.regs()
        for f in gregs.dtype.names:
            bad = np.nonzero((gregs[f] != oregs[f]).reshape(len(oregs), -1).any(axis=1))[0]
            assert bad.size == 0, f"{tag}: regs.{f} differs for sampled envs {bad[:8]}: gpu {gregs[f][bad[:4]]} oracle {oregs[f][bad[:4]]}"
        bad = np.nonzero((gram != oram).any(axis=1))[0]
        assert bad.size == 0, f"{tag}: RAM differs for sampled envs {bad[:8]}"
        if screens:
            gscr = g.get_screen(self.scr)[self.idx].cpu().numpy()
            bad = np.nonzero((gscr != o.screen()).any(axis=(1, 2)))[0]
            assert bad.size == 0, f"{tag}: screen differs for sampled envs {bad[:8]}"


def test_config2_as_stated_every_env_every_step(torch):
    """BASELINE config 2 exactly as stated: 1024 envs sharing one 4 KB ROM, per-env uniform random actions, frameskip 4,
    500 steps; RAM, regs and the 160x210 screen of EVERY env checked after EVERY step."""
    w = make_workload(2)
    g, o = mk(torch, w)
    cmp = _DevCompare(torch, g, np.arange(w.batch))
    for t0 in range(0, 500, 100):
        acts = w.actions(t0, t0 + 100); dacts = torch.from_numpy(acts).cuda()
        for t in range(100):
            g.step(dacts[t], 4); o.step(acts[t], 4, threads=NCPU)
            cmp.check(o, f"config2 step {t0 + t}")
    assert int(g.regs_host()["frame"].min()) >= 2000


def test_config3_as_stated(torch):
    """BASELINE config 3 as SURVEY G.2 states it: 16,384 envs, sticky actions, frameskip 4, 2000 steps; ALL envs checked
    against the oracle at steps 1, 10 and 100, the stratified subset e % 128 == 0 after EVERY step of the 2000."""
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    w = make_workload(3)
    idx = np.arange(0, w.batch, 128)
    g = VCS(w.roms, w.seeds, w.env_rom)
    o_all = OracleVCS(w.roms, w.seeds, w.env_rom)
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    cmp_all, cmp = _DevCompare(torch, g, np.arange(w.batch)), _DevCompare(torch, g, idx)
    for t0 in range(0, 2000, 100):
        acts = w.actions(t0, t0 + 100); dacts = torch.from_numpy(acts).cuda()
        for t in range(100):
            g.step(dacts[t], 4); o.step(acts[t][idx], 4, threads=NCPU)
            cmp.check(o, f"config3 step {t0 + t + 1}")
            if o_all is not None:
                o_all.step(acts[t], 4, threads=NCPU)
                if t0 + t + 1 in (1, 10, 100):
                    cmp_all.check(o_all, f"config3 all envs, step {t0 + t + 1}")
                if t0 + t + 1 == 100:
                    o_all.close(); o_all = None
    assert int(g.regs_host()["frame"].min()) >= 8000


def _undoc_rom(seed: int) -> bytes:
    """The paper's 38 undocumented opcode bytes (tests/golden/undocumented_opcodes.txt) mixed into ordinary code:
    NOPs of every addressing mode (their reads are real bus reads: RIOT timer, TIA collision latches, page crossings),
    LAX from RAM / ROM / through pointers, SAX into RAM and into TIA registers, USBC in binary and decimal mode."""
    r = SplitMix64(seed)

    def build(a):
        a.org(0xF000); a.op("LDX", "imm", 0xFF); a.op("TXS")
        for zp, target in ((0x90, 0xFAF0), (0x92, 0x00C0), (0x94, 0xF900)):            # pointers for (zp),Y and (zp,X)
            a.op("LDA", "imm", target & 0xFF); a.op("STA", "zp", zp); a.op("LDA", "imm", target >> 8); a.op("STA", "zp", zp + 1)
        a.label("top")
        for i in range(260):
            k = r.rnd(16)
            if k < 3: a.byte(r.choice([0x1A, 0x3A, 0x5A, 0x7A, 0xDA, 0xFA]))
            elif k < 4: a.byte(r.choice([0x80, 0x82, 0x89, 0xC2, 0xE2]), r.rnd(256))
            elif k < 5: a.byte(r.choice([0x04, 0x44, 0x64]), r.choice([r.rnd(16), 0x80 + r.rnd(128)]))          # zp: TIA read or RAM
            elif k < 6: a.byte(r.choice([0x14, 0x34, 0x54, 0x74, 0xD4, 0xF4]), r.rnd(256))
            elif k < 7:
                lo = RIOT["INTIM"] - 0x10 + r.rnd(0x20) if r.chance(1, 2) else 0xF900 + r.rnd(0x100)
                a.byte(r.choice([0x0C, 0x1C, 0x3C, 0x5C, 0x7C, 0xDC, 0xFC]), lo & 0xFF, lo >> 8)                # abs / abs,X incl. the RIOT
            elif k < 9:
                opc = r.choice([0xA7, 0xB7, 0xAF, 0xBF, 0xA3, 0xB3])
                if opc in (0xA7, 0xB7): a.byte(opc, 0x80 + r.rnd(0x60))
                elif opc in (0xAF, 0xBF): t = r.choice([0xF900 + r.rnd(0x1F0), 0x0080 + r.rnd(0x60)]); a.byte(opc, t & 0xFF, t >> 8)
                else:
                    if opc == 0xA3: a.op("LDX", "imm", r.rnd(256) if r.chance(1, 2) else r.rnd(3) * 2)     # (zp,X): the pointer cells may be anywhere in page 0
                    a.byte(opc, r.choice([0x90, 0x92, 0x94, r.rnd(256)]) if opc == 0xB3 else 0x90)
            elif k < 11:
                opc = r.choice([0x87, 0x97, 0x8F, 0x83])
                if opc in (0x87, 0x97): a.byte(opc, r.choice([0x80 + r.rnd(0x60), TIA_W[r.choice(["COLUBK", "PF1", "GRP0", "COLUPF", "ENAM0"])]]))
                elif opc == 0x8F: a.byte(opc, 0x80 + r.rnd(0x60), 0x00)
                else: a.op("LDX", "imm", r.rnd(256) if r.chance(1, 2) else r.rnd(3) * 2); a.byte(opc, 0x90)      # (zp,X) -> pointer at $90/$92/$94 or anywhere
            elif k < 12:
                if r.chance(1, 2): a.op("SED")
                a.byte(0xEB, r.rnd(256)); a.op("CLD")
            elif k < 13: a.op(r.choice(["LDX", "LDY", "LDA"]), "imm", r.rnd(4) * 2)
            elif k < 14: a.op("STA", "zp", TIA_W[r.choice(["WSYNC", "GRP1", "PF2", "HMOVE", "RESP0"])])
            elif k < 15: a.op("LDA", "imm", r.rnd(256)); a.op("STA", "abs", RIOT[r.choice(["TIM8T", "TIM64T"])])
            else: a.op(r.choice(["INX", "DEY", "CLC", "SEC", "TXA", "TAY"]))
        a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VSYNC"]); a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VSYNC"])
        a.op("JMP", "abs", "top")
    return hand_rom(build)


@pytest.mark.parametrize("seed", range(4))
def test_undocumented_opcodes(torch, seed):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    rom = _undoc_rom(3000 + seed)
    seeds = env_seeds(90 + seed, 36)
    kw = dict(max_lines=200 + 40 * seed)
    g, o = VCS([rom], seeds, **kw), OracleVCS([rom], seeds, **kw)
    for t in range(8):
        a = np.array([(t + e) % 18 for e in range(36)], np.uint8)
        g.step(torch.from_numpy(a).cuda(), 1 + t % 3); o.step(a, 1 + t % 3, threads=NCPU)
        compare(g, o, f"undoc{seed} step {t}")
    assert not (g.regs_host()["status"] & 1).any()                # none of them halts the CPU any more


def test_config4_as_stated_full_length(torch):
    """BASELINE config 4 at its full batch and full length (65,536 envs over 256 ROMs, 1000 env-steps of frameskip 4, the
    launch configuration bench.py times): one env per ROM (lane and warp varying) runs on the oracle beside the GPU;
    RAM and regs compared after every step, screens every 25 steps and at the final step (BASELINE.json: "bit-exact
    RAM/screen at the final step")."""
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    w = make_workload(4)
    idx = np.arange(256) * 256 + (np.arange(256) * 91) % 256
    g = VCS(w.roms, w.seeds, w.env_rom)
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    cmp = _DevCompare(torch, g, idx)
    for t0 in range(0, 1000, 100):
        acts = w.actions(t0, t0 + 100); dacts = torch.from_numpy(acts).cuda()
        for t in range(100):
            g.step(dacts[t], w.frameskip); o.step(acts[t][idx], w.frameskip, threads=NCPU)
            n = t0 + t + 1
            cmp.check(o, f"config4 step {n}", screens=(n % 25 == 0 or n == 1000))
    r = g.regs_host()
    assert int(r["frame"].min()) >= 4000 and (r["status"] == 0).all()


def test_block_placement_permutes_groups_not_results(torch):
    """Measured block placement: after a few plain steps of config 4 at full batch the block -> env-group
    map is a non-trivial permutation, every block has a time stamp and an SM, at most two blocks share an SM — and the
    state is what a handle with the placement switched off computes (envs are independent)."""
    from paper_2606_22447_b200 import VCS
    w = make_workload(4)
    acts = torch.from_numpy(w.actions(0, 6)).cuda()
    from paper_2606_22447_b200.binding import VCS_F_NO_BALANCE
    g = VCS(w.roms, w.seeds, w.env_rom)
    ref = VCS(w.roms, w.seeds, w.env_rom, flags=VCS_F_NO_BALANCE)
    for t in range(6):
        g.step(acts[t], 4); ref.step(acts[t], 4)
    times, perm = g.block_times()
    assert sorted(perm.tolist()) == list(range(256)) and perm.tolist() != list(range(256))
    assert (times[:, 1] > times[:, 0]).all() and np.bincount(times[:, 2].astype(np.int64)).max() <= 2
    _, perm0 = ref.block_times()
    assert perm0.tolist() == list(range(256))
    assert (g.get_ram() == ref.get_ram()).all() and (g.get_regs() == ref.get_regs()).all() and (g.get_screen() == ref.get_screen()).all()


def test_two_wave_batch_longest_first_placement(torch):
    """131,072 envs = 512 blocks on 296 block slots: the launch runs in two waves and the placement kernel orders the
    blocks longest first; a sample of envs against the oracle, and the block order must still be a permutation."""
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    w = make_workload(4, batch=131072, n_roms=256)
    idx = np.arange(64) * 2048 + (np.arange(64) * 197) % 2048
    g = VCS(w.roms, w.seeds, w.env_rom)
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    acts = w.actions(0, 6)
    for t in range(6):
        g.step(torch.from_numpy(acts[t]).cuda(), 4); o.step(acts[t][idx], 4, threads=NCPU)
    compare(g, o, "two waves", envs=idx)
    _, perm = g.block_times()
    assert sorted(perm.tolist()) == list(range(512)) and perm.tolist() != list(range(512))
