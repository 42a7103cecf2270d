"""biobeam split-step BPM hot path, B200-native (sm_100a).  See DESIGN.md."""
