"""Helpers for the -m gpu tests: run the CUDA path through the C ABI and fetch numpy results."""
import paper_2606_26089_b200 as pd


def run_gpu(card_name, ev, seed, event_base=0, debug=True, tile_events=0):
    card = pd.Card(card_name)
    dev = pd.DeviceEvents(ev)
    out = pd.DeviceOutputs(card, dev.n_events, dev.n_particles, debug=debug, tile_events=tile_events)
    pd.simulate(card, dev, out, seed, event_base)
    res = out.to_numpy()
    res["status_word"] = pd.last_status(out)
    res["launches"] = pd.last_launch_count()
    return res
