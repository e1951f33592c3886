"""Per-step parity protocol (SURVEY.md call stack 3): the CUDA step is seeded from the oracle's
prior state, every intermediate is compared element by element, and the run continues from the
ORACLE's next state."""
import numpy as np

from paper_1603_09255_b200 import workloads

INT_FIELDS = ["f", "off", "mother", "father", "dest", "zi", "alive", "captured"]


def load_initial(obj, cfg, step=0):
    for s in range(len(cfg["species"])):
        obj.write_state(s, workloads.initial_rows(cfg, s), workloads.initial_patch_start(cfg, s), step)
        if cfg["species"][s].get("separate_sexes"):
            obj.write_sex(s, workloads.initial_sex(cfg, s))


def assert_debug_equal(dg, do, species_cfg, tag=""):
    """bit-exact for integer / index / genome work, bit-exact fp32 for u01 and s (both sides take
    the decision in the same specified fp32 arithmetic, R11)."""
    assert dg["n_t"] == do["n_t"], tag
    assert dg["m_t"] == do["m_t"], tag
    if do["n_t"] == 0:      # an extinct species is skipped (its step has no intermediates); log and state are still compared
        return
    for k in INT_FIELDS:
        assert np.array_equal(dg[k], do[k]), (tag, k)
    assert np.array_equal(dg["table_len"], do["table_len"]), tag
    for t, n in enumerate(do["table_len"]):
        assert np.array_equal(dg["tables"][t, :n], do["tables"][t, :n]), (tag, "table", t)
    assert np.array_equal(dg["u01"].view(np.uint32), do["u01"].view(np.uint32)), tag
    assert np.array_equal(dg["s"].view(np.uint32), do["s"].view(np.uint32)), (tag, "s")
    assert np.array_equal(dg["offspring"], do["offspring"]), (tag, "offspring rows")
    for k in ("theta_t", "zbar_pred", "attack_n"):
        assert np.float32(dg[k]) == np.float32(do[k]), (tag, k)
    if species_cfg["fecundity"] == "captures":
        assert np.array_equal(dg["cap"], do["cap"]), (tag, "cap")
    if species_cfg.get("adult_survival", 0.0) > 0.0:   # R18: the adults' own survival
        assert np.array_equal(dg["a_alive"], do["a_alive"]), (tag, "a_alive")
        assert np.array_equal(dg["a_u"].view(np.uint32), do["a_u"].view(np.uint32)), (tag, "a_u")
        assert np.array_equal(dg["a_s"].view(np.uint32), do["a_s"].view(np.uint32)), (tag, "a_s")


    if species_cfg.get("separate_sexes"):               # R21: sex at birth
        assert np.array_equal(dg["sex_off"], do["sex_off"]), (tag, "sex_off")
    if species_cfg.get("mate_skew", 0.0) != 0.0 or species_cfg.get("separate_sexes"):        # R19: the integer mating weights' running sum
        assert np.float32(dg["zbar_self"]) == np.float32(do["zbar_self"]), (tag, "zbar_self")
        assert np.array_equal(dg["mate_cum"], do["mate_cum"]), (tag, "mate_cum")
    if species_cfg.get("mother_skew", 0.0) != 0.0:                                           # R24: the mothering weights' running sum
        assert np.float32(dg["zbar_self"]) == np.float32(do["zbar_self"]), (tag, "zbar_self")
        assert np.array_equal(dg["mom_cum"], do["mom_cum"]), (tag, "mom_cum")


def assert_state_equal(sim, orc, cfg, tag=""):
    for s in range(len(cfg["species"])):
        rg, pg, zg = sim.read_state(s)
        ro, po, zo = orc.read_state(s)
        assert rg.shape == ro.shape, (tag, s, rg.shape, ro.shape)
        assert np.array_equal(rg, ro), (tag, s, "rows")
        assert np.array_equal(pg, po), (tag, s, "patch_start")
        assert np.array_equal(zg, zo), (tag, s, "zi")
        if cfg["species"][s].get("separate_sexes"):
            assert np.array_equal(sim.read_sex(s), orc.read_sex(s)), (tag, s, "sex")


def assert_logs_equal(lg, lo, tag=""):
    assert len(lg) == len(lo), tag
    for a, b in zip(lg, lo):
        assert a == b, (tag, a, b)


def per_step_parity(oracle_mod, binding, cfg, steps, debug=True):
    """Runs `steps` steps; before each, the CUDA sim is re-seeded from the oracle's state."""
    orc = oracle_mod.Oracle(cfg)
    load_initial(orc, cfg)
    sim = binding.Sim(cfg, debug=debug)
    ties = 0
    for t in range(steps):
        for s in range(len(cfg["species"])):
            rows, ps, _ = orc.read_state(s)
            sim.write_state(s, rows, ps if sim.P > 1 else None, t)
            if cfg["species"][s].get("separate_sexes"):
                sim.write_sex(s, orc.read_sex(s))
        orc.step(1)
        sim.step(1)
        for s in range(len(cfg["species"])):
            if debug:
                assert_debug_equal(sim.read_debug(s), orc.debug(s), cfg["species"][s], tag="step %d species %d" % (t, s))
            lg, lo = sim.read_log(s)[-1], orc.log(s)[-1]
            assert lg == lo, (t, s, lg, lo)
            ties += lo["near_ties"]
        assert_state_equal(sim, orc, cfg, tag="after step %d" % t)
        assert sim.status() == orc.flags
    sim.close()
    return ties
