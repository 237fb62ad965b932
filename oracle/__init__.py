"""CPU oracle of the Hough fill + peak search (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It never imports the CUDA package, and the CUDA package never imports it.
"""
from .ht_oracle import (MERGED_DTYPE, OracleBinning, oracle_fill, oracle_fill_batch, oracle_match_truth, oracle_merge_ridges,
                        oracle_peaks, oracle_peaks_batch, oracle_tables, oracle_tracks, oracle_votes, PEAK_DTYPE, TRUTH_DTYPE)

__all__ = ["MERGED_DTYPE", "OracleBinning", "oracle_fill", "oracle_fill_batch", "oracle_match_truth", "oracle_merge_ridges",
           "oracle_peaks", "oracle_peaks_batch", "oracle_tables", "oracle_tracks", "oracle_votes", "PEAK_DTYPE", "TRUTH_DTYPE"]
