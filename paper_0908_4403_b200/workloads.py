"""The synthetic workloads of BASELINE.json `configs` as plain data (no arithmetic).

Shared by bench.py and tests/: both the CUDA generator (heget_gen_events) and the oracle's
generator (oracle.gen_events) are driven from these parameters; each side implements the
generation itself."""

# mode names match include/heget.h HEGET_GEN_* and oracle.MODE_*
FIXED, LOGUNIFORM, TOYPDF = 0, 1, 2

PT_CUT, ETA_CUT, DR_CUT = 20.0, 2.5, 0.4   # eq. (9)
ALPHA, Q_U = 1.0 / 128.0, 2.0 / 3.0        # DESIGN.md reading R2
GEV2_TO_FB = 0.3893793721e12               # 1 GeV^-2 in fb (reading R17)

CONFIGS = {
    # name: n photons, N events, generation mode and parameters, seed, oracle subset size
    "2gamma": dict(n=2, N=1 << 16, mode=FIXED, a=1000.0, b=0.0, y_max=0.0, apply_cuts=False, seed=1,
                   oracle_events=1 << 16),
    # 3 and 5 photons are not BASELINE.json configs: same generation scheme, for the per-n report of bench.py
    "3gamma": dict(n=3, N=1 << 20, mode=LOGUNIFORM, a=150.0, b=2500.0, y_max=1.5, apply_cuts=True, seed=1,
                   oracle_events=1 << 16),
    "4gamma": dict(n=4, N=1 << 20, mode=LOGUNIFORM, a=200.0, b=3000.0, y_max=1.5, apply_cuts=True, seed=1,
                   oracle_events=1 << 14),
    "5gamma": dict(n=5, N=1 << 20, mode=LOGUNIFORM, a=300.0, b=4000.0, y_max=1.5, apply_cuts=True, seed=1,
                   oracle_events=2048),
    "6gamma": dict(n=6, N=1 << 20, mode=LOGUNIFORM, a=400.0, b=5000.0, y_max=1.5, apply_cuts=True, seed=1,
                   oracle_events=256),
    "7gamma": dict(n=7, N=1 << 18, mode=LOGUNIFORM, a=500.0, b=6000.0, y_max=1.5, apply_cuts=True, seed=1,
                   oracle_events=4096),
    "8gamma": dict(n=8, N=1 << 16, mode=TOYPDF, a=14000.0, b=0.0, y_max=0.0, apply_cuts=True, seed=1,
                   oracle_events=512),
}
ORDER = ["2gamma", "3gamma", "4gamma", "5gamma", "6gamma", "7gamma", "8gamma"]
BASELINE_CONFIGS = ["2gamma", "4gamma", "6gamma", "7gamma", "8gamma"]   # BASELINE.json `configs`, in its order


def shard_range(n_events, rank, world_size):
    """Contiguous range [first, first+count) of global event indices owned by `rank`."""
    base, rem = divmod(n_events, world_size)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)
