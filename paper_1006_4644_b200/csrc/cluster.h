// cluster.h -- host-side trigger clustering: "Reduce the [c(t_0)] set, in order to detect
// local maximum"; "The clusterization phase is made only by CPU.  This chose permits us to hide
// this computing part behind the next iteration".  Plain C++ on the host, no CUDA.
//
// Reading A24 (the paper gives no rule and no window): above-threshold samples of ONE template are
// chained into an event while consecutive ones are at most `window` samples apart, the segment taken as a circle
// (the filter output is circular, A11); an event is reported as its sample of largest SNR, the smallest sample index
// among equal maxima; events come out ordered by (template, that sample).
//
// This is the efficient form for a list already sorted by (template, sample) -- one scan with a running maximum and
// a wrap-around join per template; the test oracle's twin states the pairwise definition instead.
#pragma once
#include <stdint.h>
#include <vector>

namespace cbmf {

struct HostTrig { int32_t template_idx; int32_t sample_idx; float snr; float phase; };   // = cbmf_trigger

inline bool trig_better(const HostTrig& a, const HostTrig& b)      // a beats b as the representative of an event
{
    return a.snr > b.snr || (a.snr == b.snr && a.sample_idx < b.sample_idx);
}

// Events of trig[0..n) (sorted strictly by (template_idx, sample_idx), samples in [0, n_samples)) appended to `out`.
// Returns false if the list is not sorted or a sample is out of range.
inline bool cluster_sorted(const HostTrig* trig, int64_t n, int64_t n_samples, int64_t window, std::vector<HostTrig>& out)
{
    int64_t i = 0;
    while (i < n) {
        const int32_t tmpl = trig[i].template_idx;
        const size_t first_event = out.size();
        const int32_t first_sample = trig[i].sample_idx;
        HostTrig best = trig[i];
        int32_t prev = trig[i].sample_idx;
        if (tmpl < 0 || prev < 0 || prev >= n_samples) return false;
        ++i;
        for (; i < n && trig[i].template_idx == tmpl; ++i) {
            const int32_t s = trig[i].sample_idx;
            if (s <= prev || s >= n_samples) return false;
            if ((int64_t)s - prev > window) { out.push_back(best); best = trig[i]; }
            else if (trig_better(trig[i], best)) best = trig[i];
            prev = s;
        }
        if (i < n && trig[i].template_idx < tmpl) return false;
        // `best` is the still open last event.  Around the circle it joins the first event of this template when the gap
        // from the last sample to the first one is within the window (and the two are not the same event).
        if (out.size() > first_event && (int64_t)first_sample + n_samples - prev <= window) {
            HostTrig& head = out[first_event];
            if (trig_better(best, head)) {
                // the representative lies in the tail part: it sorts after every other event of this template
                out.erase(out.begin() + (std::ptrdiff_t)first_event);
                out.push_back(best);
            }
        } else {
            out.push_back(best);
        }
    }
    return true;
}

}  // namespace cbmf
