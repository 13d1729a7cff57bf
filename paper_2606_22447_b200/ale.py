"""ALE-style vector environment over libvcsb200.

PAPER.md L167: "the standard ALE boot (60 no-op frames plus four resets) and then a fixed action stream";
Table 8: "Boot sequence: 60 NOOP + 4 RESET frames; episode-start randomization: 0-30 random NOOPs
(Mnih-style)".  Everything the consoles do runs in the library (vcs_boot, vcs_step, vcs_step_masked,
vcs_set_switches); this class only sequences those calls, draws the NOOP-start counts (seeded, on the device) and
keeps the episode step counters.  Per-game reward / terminal logic needs the games and is out of scope: the caller
passes its own `done` mask (e.g. computed from `ram()`), and the envs it names are re-booted in place while the
others carry on — per-env auto-reset.  With `amortised=True` (default when the boot frame counts are multiples of
`frameskip`) the re-boot is vcs_auto_reset: the env is reset and armed, its boot runs inside the batch's following
vcs_step calls (no extra launches), and `booting()` says which envs do not yet follow the agent."""
from __future__ import annotations

from .binding import VCS


class AleVecEnv:
    def __init__(self, roms, seeds, env_rom=None, frameskip=4, noop_max=30, boot_noop_frames=60, boot_reset_frames=4,
                 max_episode_steps=None, start_seed=0, amortised=None, **config):
        self.vcs = VCS(roms, seeds, env_rom, **config)
        t = self.torch = self.vcs.torch
        self.batch, self.device = self.vcs.batch, self.vcs.device
        self.frameskip, self.noop_max = int(frameskip), int(noop_max)
        self.boot_noop_frames, self.boot_reset_frames = int(boot_noop_frames), int(boot_reset_frames)
        self.max_episode_steps = max_episode_steps
        assert 0 <= self.noop_max <= 255
        divisible = self.boot_noop_frames % self.frameskip == 0 and self.boot_reset_frames % self.frameskip == 0
        self.amortised = divisible if amortised is None else bool(amortised)
        assert divisible or not self.amortised, "amortised boot needs boot frame counts that are multiples of frameskip"
        self._gen = t.Generator(device=self.device); self._gen.manual_seed(int(start_seed))
        self.episode_steps = t.zeros(self.batch, dtype=t.int32, device=self.device)
        self.episodes = t.zeros(self.batch, dtype=t.int32, device=self.device)

    # ---- episode starts
    def _draw_starts(self):
        t = self.torch
        return t.randint(0, self.noop_max + 1, (self.batch,), generator=self._gen, device=self.device, dtype=t.int32).to(t.uint8)

    def reset(self, mask=None, noop_starts=None):
        """Boot the envs with mask != 0 (None = all): reset, NOOP frames, RESET-switch frames, 0..noop_max NOOP steps
        (drawn here unless `noop_starts` uint8[batch] is given).  Returns the starts used."""
        starts = self._draw_starts() if noop_starts is None else noop_starts
        self.last_starts = starts
        self.vcs.boot(mask, self.boot_noop_frames, self.boot_reset_frames, starts if self.noop_max > 0 else None,
                      self.noop_max, self.frameskip)
        if mask is None:
            self.episode_steps.zero_(); self.episodes += 1
        else:
            m = mask != 0
            self.episode_steps.masked_fill_(m, 0); self.episodes += m.to(self.episodes.dtype)
        return starts

    # ---- one agent step
    def step(self, actions, done=None):
        """vcs_step with `frameskip`; then re-boot the envs the caller marks `done` (uint8/bool [batch], from its own
        game logic) and those that hit max_episode_steps.  Returns the uint8[batch] mask of the envs that were re-booted
        (their observation is the first one of the new episode)."""
        t = self.torch
        # an env that is still running its (amortised) boot ignores the agent in this step: the step does not count
        # towards its episode, and a `done` the caller computed from its RAM meanwhile does not re-arm it
        playing = (self.vcs.get_booting() == 0) if self.amortised else None
        self.vcs.step(actions, self.frameskip)
        self.episode_steps += 1 if playing is None else playing.to(self.episode_steps.dtype)
        over = None
        if done is not None:
            over = (done != 0) if playing is None else ((done != 0) & playing)
        if self.max_episode_steps is not None:
            trunc = self.episode_steps >= int(self.max_episode_steps)
            over = trunc if over is None else (over | trunc)
        if over is None:
            return t.zeros(self.batch, dtype=t.uint8, device=self.device)
        mask = over.to(t.uint8).contiguous()
        if bool(mask.any()):
            if self.amortised:
                self.last_starts = self._draw_starts()
                self.vcs.auto_reset(mask, self.boot_noop_frames // self.frameskip, self.boot_reset_frames // self.frameskip,
                                    self.last_starts if self.noop_max > 0 else None, self.noop_max)
                self.episode_steps.masked_fill_(over, 0); self.episodes += over.to(self.episodes.dtype)
            else:
                self.reset(mask)
        return mask

    def booting(self, out=None):
        """uint8[batch]: boot steps each env still has to run before it follows the agent (0 = playing)."""
        return self.vcs.get_booting(out)

    # ---- observations (device tensors)
    def screen(self, out=None):
        return self.vcs.get_screen(out)

    def ram(self, out=None):
        return self.vcs.get_ram(out)

    def set_switches(self, switches=None):
        self.vcs.set_switches(switches)

    def close(self):
        self.vcs.close()
