"""Parameter scans on synthetic events (the paper's Fig. 10, 11, 12).

  python -m paper_2402_14670_b200.scan [--events 4000] [--steps 20] [--out profiles/r1_scans.md]

* n_window scan (Fig. 10): efficiency for particles with p > 5 GeV and pT > 1 GeV, ghost rate and
  events/s against the cap on the hits per search window, (a) with the window tolerances fixed and (b) with the
  x tolerance scaled in proportion ("the n_window variable is proportional to the search window size").
* occupancy scan (Fig. 11-12): the same quantities against the event occupancy (tracks, fake seeds
  and noise hits scaled together - the stand-in for the number of pp collisions per event).

* concurrent streams: the same batch cut into event ranges that run on several CUDA streams at once.

Everything runs through the C ABI on cuda:0 (no CPU fallback); efficiencies use the generator's truth
(`truth.evaluate`, the paper's 70 % matching rule).  Prints a markdown report.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np


def _kinematic_mask(batch, p_min=5.0, pt_min=1.0):
    """True tracks with p > 5 GeV and pT > 1 GeV (the denominator of the paper's Fig. 10)."""
    p = 1.0 / np.abs(batch.trk_qop)
    s2 = batch.trk_tx ** 2 + batch.trk_ty ** 2
    pt = p * np.sqrt(s2 / (1.0 + s2))
    return (p > p_min) & (pt > pt_min)


def measure(binding, truth, G, P, batch, steps: int):
    import torch
    lf = binding.LookingForward(G, P, batch.n_events, batch.n_seeds, batch.n_hits)
    db = binding.DeviceBatch(batch)
    out = binding.TrackBuffers(batch.n_seeds, batch.n_events, db.device)
    stream = torch.cuda.current_stream()
    for _ in range(3):
        lf.run(db, out, stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        lf.run(db, out, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    r = out.to_numpy()
    lf.close()
    ev = truth.evaluate(batch, r.hit_idx, r.n_hits)
    rec = truth.reconstructible(batch) & _kinematic_mask(batch)
    found = np.zeros(batch.n_tracks, bool)
    found[ev.matched_track[ev.matched_track >= 0]] = True
    return dict(ms=ms, events_per_s=batch.n_events / (ms * 1e-3), seeds_per_s=batch.n_seeds / (ms * 1e-3),
                eff_all=ev.efficiency, eff_kin=float(found[rec].mean()) if rec.any() else 0.0, ghost=ev.ghost_rate,
                tracks=r.n_tracks)


def measure_streams(binding, G, P, batch, n_streams: int, steps: int):
    """The batch cut into `n_streams` event ranges, each with its own handle and CUDA stream, all in flight together
    (the paper's way of filling the GPU: several streams, each with its own batch of events)."""
    import torch
    from . import sharding
    ranges = sharding.event_ranges(batch.seed_offsets, n_streams)
    parts = [batch.slice_events(e0, e1) for e0, e1 in ranges]
    lfs = [binding.LookingForward(G, P, p.n_events, p.n_seeds, p.n_hits) for p in parts]
    dbs = [binding.DeviceBatch(p) for p in parts]
    outs = [binding.TrackBuffers(p.n_seeds, p.n_events, dbs[0].device) for p in parts]
    streams = [torch.cuda.Stream() for _ in parts]
    main = torch.cuda.current_stream()

    def step():
        for lf, db, out, st in zip(lfs, dbs, outs, streams):
            lf.run(db, out, st)
    for _ in range(3):
        step()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(main)
    for st in streams:
        st.wait_stream(main)
    for _ in range(steps):
        step()
    for st in streams:
        main.wait_stream(st)
    e1.record(main)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    tracks = sum(int(o.n_tracks.cpu()[0]) for o in outs)
    for lf in lfs:
        lf.close()
    return dict(ms=ms, events_per_s=batch.n_events / (ms * 1e-3), tracks=tracks)


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--events", type=int, default=4000, help="events of the Run-3-like batch (configs[1] recipe)")
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--out", default=None, help="also write the report to this file")
    ap.add_argument("--sections", default="window,occupancy,streams", help="comma list of window, occupancy, streams")
    args = ap.parse_args(argv)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("scan.py needs a CUDA device (there is no CPU fallback)")
    from . import binding, datagen, truth
    G = datagen.toy_geometry()
    lines = ["# Scans on synthetic events (B200, through the C ABI)", "",
             f"Command: `python -m paper_2402_14670_b200.scan --events {args.events} --steps {args.steps}`.",
             "Efficiency (p > 5 GeV, pT > 1 GeV) is measured against reconstructible particles of that kinematic range;",
             "'all' against every reconstructible particle (p > 2 GeV); matching rule of PAPER.md:100-102.", ""]

    base = datagen.generate(datagen.with_overrides(datagen.CONFIGS[1], seed=2001), n_events=args.events)
    hits_per_seg = base.n_hits / (base.n_events * 24)

    def table(title, rows, first_col):
        lines.extend([f"## {title}", "", f"| {first_col} | ms/step | events/s | seeds/s | eff (p>5, pT>1) | eff (all) | ghost rate | tracks |",
                      "|---|---|---|---|---|---|---|---|"])
        for label, m in rows:
            lines.append(f"| {label} | {m['ms']:.3f} | {m['events_per_s'] / 1e6:.2f} M | {m['seeds_per_s'] / 1e6:.0f} M | "
                         f"{100 * m['eff_kin']:.2f} % | {100 * m['eff_all']:.2f} % | {100 * m['ghost']:.2f} % | {m['tracks']} |")
        lines.append("")

    sections = set(args.sections.split(","))
    P0, P1 = datagen.default_params(), datagen.no_ut_params()
    if "window" in sections:
        scan_window(binding, truth, datagen, G, base, args, table, hits_per_seg)
    if "occupancy" in sections:
        scan_occupancy(binding, truth, datagen, G, args, table)
    if "streams" in sections:
        scan_streams(binding, datagen, G, args, lines)
    report = "\n".join(lines)
    print(report)
    if args.out:
        with open(args.out, "w") as fh:
            fh.write(report + "\n")
    return 0


def scan_window(binding, truth, datagen, G, base, args, table, hits_per_seg):
    # ---- n_window scans (Fig. 10)
    P0 = datagen.default_params()
    rows = [(str(nw), measure(binding, truth, G, dict(P0, n_window=nw), base, args.steps)) for nw in (4, 8, 12, 16, 24, 32, 48, 64)]
    table(f"n_window scan, with-UT tuning, window tolerances fixed ({args.events} events, {hits_per_seg:.0f} hits per layer half; "
          "n_window > 32 runs the wide kernels)", rows, "n_window")
    rows = []
    for nw in (8, 16, 24, 32, 48, 64):
        f = nw / 32.0
        P = dict(P0, n_window=nw, xtol_base=P0["xtol_base"] * f, xtol_inv_p=P0["xtol_inv_p"] * f, uv_half_width=P0["uv_half_width"] * f)
        rows.append((f"{nw} (tolerances x {f:.2f})", measure(binding, truth, G, P, base, args.steps)))
    table("n_window scan, with-UT tuning, window tolerances scaled in proportion to n_window", rows, "n_window")
    P1 = datagen.no_ut_params()
    rows = [(str(nw), measure(binding, truth, G, dict(P1, n_window=nw), base, args.steps)) for nw in (16, 32, 48, 64)]
    table("n_window scan, no-UT tuning (PAPER.md:323: 64)", rows, "n_window")



def scan_occupancy(binding, truth, datagen, G, args, table):
    # ---- occupancy scan (Fig. 11, 12)
    P0, P1 = datagen.default_params(), datagen.no_ut_params()
    rows_ut, rows_no = [], []
    for f in (0.25, 0.5, 1.0, 1.5, 2.0, 3.0):
        c = datagen.CONFIGS[1]
        cfg = datagen.with_overrides(c, seed=2100 + int(100 * f), true_mean=c.true_mean * f, fake_mean=c.fake_mean * f,
                                     noise_mean=c.noise_mean * f)
        b = datagen.generate(cfg, n_events=max(200, int(args.events / max(f, 0.5))))
        label = f"x {f:g} ({b.n_seeds / b.n_events:.0f} seeds, {b.n_hits / b.n_events:.0f} hits per event)"
        rows_ut.append((label, measure(binding, truth, G, P0, b, args.steps)))
        rows_no.append((label, measure(binding, truth, G, P1, b, args.steps)))
    table("occupancy scan, with-UT tuning (x 1 = BASELINE.json configs[1] occupancy)", rows_ut, "occupancy")
    table("occupancy scan, no-UT tuning", rows_no, "occupancy")


def scan_streams(binding, datagen, G, args, lines):
    # ---- concurrent streams
    P0 = datagen.default_params()
    big = datagen.generate(datagen.with_overrides(datagen.CONFIGS[1], seed=2001), n_events=5 * args.events)
    lines.extend([f"## concurrent streams, with-UT tuning ({big.n_events} events cut into equal-seed-count ranges, one handle and one stream each)", "",
                  "| streams | ms/step | events/s | tracks |", "|---|---|---|---|"])
    for ns in (1, 2, 4, 8):
        m = measure_streams(binding, G, P0, big, ns, args.steps)
        lines.append(f"| {ns} | {m['ms']:.3f} | {m['events_per_s'] / 1e6:.2f} M | {m['tracks']} |")
    lines.append("")


if __name__ == "__main__":
    sys.exit(main())
