"""The metric of the paper and the bytes-per-site model of the roofline.

SUPS ("Site Updates Per Second") = fluid sites x time steps / wall seconds; this
reproduces Table III of the paper from Table II to the integer (
tests/golden/paper_tables_II_III.txt).
"""


def sups(n_sites: int, steps: int, seconds: float) -> float:
    return float(n_sites) * float(steps) / float(seconds)


def msups(n_sites: int, steps: int, seconds: float) -> float:
    return sups(n_sites, steps, seconds) / 1.0e6


# Algorithmic bytes per site update: 15
# populations read + 15 written + 14 int32 table entries; A-A reads the table on odd steps only.
BYTES_PER_SITE = {
    ("two_lattice", "f64"): 296.0,
    ("aa", "f64"): 268.0,
    ("two_lattice", "f32"): 176.0,
    ("aa", "f32"): 148.0,
}


def algorithmic_bytes_per_site(scheme: str, store: str, n_q: int = 15) -> float:
    """Q populations read + Q written + (Q - 1) int32 table entries (A-A: on odd steps only)."""
    if n_q == 15:
        return BYTES_PER_SITE[(scheme, store)]
    pop = 8.0 if store == "f64" else 4.0
    table = 4.0 * (n_q - 1)
    return 2.0 * n_q * pop + (table if scheme == "two_lattice" else table / 2.0)


def moved_bytes_per_site(scheme: str, store: str, n_q: int = 15, records: bool = True,
                         sentinel_fraction: float = 0.0, phase: str = "step",
                         bfl_site_fraction: float = 0.0) -> float:
    """Bytes one site update of the selected variant really has to move (the model ncu's DRAM
    counters are compared with): Q populations read + Q written, the links in the form the
    kernel reads them -- 16-byte run-length records per (warp, link), i.e. (Q - 1) / 2 bytes
    per site, plus the int32 table rows of the sentinel records; or the whole table -- and one
    iolet bit per site. ``phase``: "step" (A-A: mean of the even and odd kernels), "even", "odd".
    With interpolated (BFL) walls every kernel also reads one {bits, rank} word per 32 sites and,
    for the ``bfl_site_fraction`` of the sites that carry an interpolated link, one row of
    (Q - 1) / 2 coefficients + a member word, padded to an even count of doubles (64 B / 80 B).
    """
    pop = 8.0 if store == "f64" else 4.0
    bfl = 0.0
    if bfl_site_fraction > 0.0:
        bfl = 8.0 / 32.0 + bfl_site_fraction * 8.0 * (((n_q - 1) // 2 + 2) // 2 * 2)
    links = (16.0 * (n_q - 1) / 32.0 + sentinel_fraction * 4.0 * (n_q - 1)) if records \
        else 4.0 * (n_q - 1)
    base = 2.0 * n_q * pop + 4.0 / 32.0 + bfl
    if scheme == "two_lattice" or phase == "odd":
        return base + links
    if phase == "even":
        return base
    return base + links / 2.0
